// Host-side acceleration-structure build: binned-SAH BVH2, collapsed to a BVH8, children placed in octant
// slots, child boxes quantised to 8 bits per plane (80-byte nodes, dr_types.h), emitted breadth-first so that
// the top levels are contiguous (they stay in L1 / L2; staging them in shared memory was measured in round 1 and
// removed: profiles/r01f_k_trace_full.md, step r01e).
// The paper uses a hardware ray-tracing pipeline; B200 has no RT cores, so the closest-hit
// query of row a4 runs in software over this structure.  The compressed wide node with octant-ordered
// traversal follows the published idea of Ylitie, Karras and Laine (HPG 2017), restated here from scratch.
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
  uint32_t first = 0, count = 0;  // range into `order`; count != 0 marks a BVH2 leaf
  uint32_t refs = 0;              // references in the subtree = order[first, first + refs)
};

constexpr int kBins = 32;
#ifndef DR_SPLIT_BUDGET
#define DR_SPLIT_BUDGET 1.0   // extra references per triangle the pre-splitting may create
#endif

struct Builder {
  const std::vector<Box>& tb;
  const std::vector<float>& cen;  // 3 per triangle
  std::vector<uint32_t> order;
  std::vector<Node2> nodes;
  uint32_t leaf_max = kMaxLeafTris;   // 1 when the optimal collapse decides the leaves

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
    nodes[me].refs = count;
    if (count <= leaf_max) return me;
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

// Reference splitting before the build ("early split clipping", restated from the published idea of Ernst and
// Greiner 2007 / Karras and Aila 2013): a triangle whose bounding box is much larger than the triangle itself (long,
// thin, rotated: the cylinder and gear meshes of configs[3]) is cut by axis-aligned planes into several references,
// each with the tight box of its clipped piece.  All references of a triangle point at the same triangle, so the
// closest hit is unchanged; only the boxes the traversal sees get tighter.  The worst references (largest box area in
// excess of the piece's own projected area) are split first until the budget of extra references is used up.
struct Ref {
  Box box;
  uint32_t tri;
};

struct Poly {
  int n = 0;
  double p[10][3];
};

void clip_poly(const Poly& in, int axis, double plane, bool keep_low, Poly& out) {
  out.n = 0;
  for (int i = 0; i < in.n; ++i) {
    const double* a = in.p[i];
    const double* b = in.p[(i + 1) % in.n];
    const double da = keep_low ? plane - a[axis] : a[axis] - plane, db = keep_low ? plane - b[axis] : b[axis] - plane;
    if (da >= 0.0 && out.n < 10) { for (int k = 0; k < 3; ++k) out.p[out.n][k] = a[k]; ++out.n; }
    if ((da > 0.0 && db < 0.0) || (da < 0.0 && db > 0.0)) {
      const double t = da / (da - db);
      if (out.n < 10) {
        for (int k = 0; k < 3; ++k) out.p[out.n][k] = a[k] + t * (b[k] - a[k]);
        out.p[out.n][axis] = plane;
        ++out.n;
      }
    }
  }
}

Box poly_box(const Poly& q) {
  Box b;
  for (int i = 0; i < q.n; ++i) {
    const float f[3] = {(float)q.p[i][0], (float)q.p[i][1], (float)q.p[i][2]};
    // round outwards: the float box must contain the double-precision piece
    float lo[3], hi[3];
    for (int k = 0; k < 3; ++k) {
      lo[k] = (double)f[k] > q.p[i][k] ? std::nextafter(f[k], -FLT_MAX) : f[k];
      hi[k] = (double)f[k] < q.p[i][k] ? std::nextafter(f[k], FLT_MAX) : f[k];
    }
    b.grow(lo);
    b.grow(hi);
  }
  return b;
}

double poly_ideal_area(const Poly& q) {  // surface area of the tightest possible box of a flat piece: 2 * sum of projections
  double n[3] = {0, 0, 0};
  for (int i = 1; i + 1 < q.n; ++i) {
    const double u[3] = {q.p[i][0] - q.p[0][0], q.p[i][1] - q.p[0][1], q.p[i][2] - q.p[0][2]};
    const double v[3] = {q.p[i + 1][0] - q.p[0][0], q.p[i + 1][1] - q.p[0][1], q.p[i + 1][2] - q.p[0][2]};
    n[0] += u[1] * v[2] - u[2] * v[1]; n[1] += u[2] * v[0] - u[0] * v[2]; n[2] += u[0] * v[1] - u[1] * v[0];
  }
  return std::fabs(n[0]) + std::fabs(n[1]) + std::fabs(n[2]);  // 2 * (1/2) * |n| components
}

void presplit(const float* verts, const uint32_t* idx, uint32_t nt, double budget_factor, std::vector<Ref>& refs) {
  struct Piece { Poly poly; Box box; uint32_t tri; };
  typedef std::pair<double, uint32_t> Key;  // (excess area, piece index): worst first
  std::priority_queue<Key> pq;
  std::vector<Piece> pool;
  refs.clear();
  refs.reserve((size_t)(nt * (1.0 + budget_factor)) + 8);
  std::vector<double> excess(nt);
  double total_area = 0.0;
  Poly tp;
  tp.n = 3;
  auto load = [&](uint32_t t, Box& box) {
    box = Box();
    for (int k = 0; k < 3; ++k) {
      for (int a = 0; a < 3; ++a) tp.p[k][a] = verts[3 * idx[3 * t + k] + a];
      box.grow(&verts[3 * idx[3 * t + k]]);
    }
  };
  for (uint32_t t = 0; t < nt; ++t) {
    Box box;
    load(t, box);
    const double ideal = poly_ideal_area(tp);
    excess[t] = (double)box.area() - ideal;
    total_area += ideal;
  }
  // pieces whose excess is below a share of the mean triangle area are never worth a split
  const double floor_excess = 0.5 * total_area / std::max(1u, nt);
  long budget = (long)(budget_factor * nt);
  for (uint32_t t = 0; t < nt; ++t) {
    Box box;
    load(t, box);
    if (budget > 0 && excess[t] > floor_excess) {
      pq.push(Key(excess[t], (uint32_t)pool.size()));
      pool.push_back({tp, box, t});
    } else {
      refs.push_back({box, t});
    }
  }
  while (!pq.empty()) {
    const Key key = pq.top();
    pq.pop();
    const Piece it = pool[key.second];
    if (budget <= 0 || key.first <= floor_excess) { refs.push_back({it.box, it.tri}); continue; }
    int axis = 0;
    float ext = -1.f;
    for (int a = 0; a < 3; ++a) if (it.box.hi[a] - it.box.lo[a] > ext) { ext = it.box.hi[a] - it.box.lo[a]; axis = a; }
    const double plane = 0.5 * ((double)it.box.lo[axis] + (double)it.box.hi[axis]);
    Piece lo, hi;
    clip_poly(it.poly, axis, plane, true, lo.poly);
    clip_poly(it.poly, axis, plane, false, hi.poly);
    if (lo.poly.n < 3 || hi.poly.n < 3) { refs.push_back({it.box, it.tri}); continue; }
    lo.tri = hi.tri = it.tri;
    lo.box = poly_box(lo.poly);
    hi.box = poly_box(hi.poly);
    for (int a = 0; a < 3; ++a) {  // pieces never leave the parent's box
      lo.box.lo[a] = std::max(lo.box.lo[a], it.box.lo[a]); lo.box.hi[a] = std::min(lo.box.hi[a], it.box.hi[a]);
      hi.box.lo[a] = std::max(hi.box.lo[a], it.box.lo[a]); hi.box.hi[a] = std::min(hi.box.hi[a], it.box.hi[a]);
    }
    --budget;
    pool[key.second] = lo;  // reuse the parent's entry
    pq.push(Key((double)lo.box.area() - poly_ideal_area(lo.poly), key.second));
    pq.push(Key((double)hi.box.area() - poly_ideal_area(hi.poly), (uint32_t)pool.size()));
    pool.push_back(hi);
  }
}

// Places up to eight children in the octant slots: child c goes to the free slot s that maximises
// dot(centre(c) - centre(node), corner(s)), greedily over all (child, slot) pairs.
void assign_slots(const std::vector<Node2>& n2, const uint32_t* kids, int nk, int* slot_of) {
  Box nb;
  for (int i = 0; i < nk; ++i) nb.grow(n2[kids[i]].box);
  float score[8][8];
  for (int i = 0; i < nk; ++i) {
    const Box& b = n2[kids[i]].box;
    float off[3];
    for (int a = 0; a < 3; ++a) off[a] = 0.5f * (b.lo[a] + b.hi[a]) - 0.5f * (nb.lo[a] + nb.hi[a]);
    for (int s = 0; s < 8; ++s)
      score[i][s] = ((s & 4) ? off[0] : -off[0]) + ((s & 2) ? off[1] : -off[1]) + ((s & 1) ? off[2] : -off[2]);
  }
  bool child_done[8] = {false}, slot_used[8] = {false};
  for (int round = 0; round < nk; ++round) {
    int bi = -1, bs = -1;
    float best = -FLT_MAX;
    for (int i = 0; i < nk; ++i) {
      if (child_done[i]) continue;
      for (int s = 0; s < 8; ++s)
        if (!slot_used[s] && score[i][s] > best) { best = score[i][s]; bi = i; bs = s; }
    }
    child_done[bi] = true;
    slot_used[bs] = true;
    slot_of[bi] = bs;
  }
}

}  // namespace

static double g_split_budget = DR_SPLIT_BUDGET;
#ifndef DR_COLLAPSE_OPTIMAL
#define DR_COLLAPSE_OPTIMAL 1
#endif
static bool g_optimal_collapse = DR_COLLAPSE_OPTIMAL != 0;
#ifndef DR_COLLAPSE_COST_TRI
#define DR_COLLAPSE_COST_TRI 0.4
#endif
static float kCostNode = 1.0f, kCostTri = (float)(DR_COLLAPSE_COST_TRI);   // relative cost of a BVH8 node test and of a triangle test in the collapse
void set_split_budget(double extra_refs_per_triangle) { g_split_budget = extra_refs_per_triangle; }
void set_collapse(bool optimal, float cost_node, float cost_tri) { g_optimal_collapse = optimal; kCostNode = cost_node; kCostTri = cost_tri; }

void build_bvh8(const float* verts, uint32_t nv, const uint32_t* idx, uint32_t nt, const uint32_t* tri_mat, BuiltBvh& out) {
  (void)nv;
  std::vector<Ref> refs;
  presplit(verts, idx, nt, g_split_budget, refs);
  const uint32_t nr = (uint32_t)refs.size();
  std::vector<Box> tb(nr);
  std::vector<float> cen(3 * (size_t)nr);
  Box scene;
  for (uint32_t t = 0; t < nr; ++t) {
    tb[t] = refs[t].box;
    for (int a = 0; a < 3; ++a) cen[3 * t + a] = 0.5f * (tb[t].lo[a] + tb[t].hi[a]);
    scene.grow(tb[t]);
  }
  const float dx = scene.hi[0] - scene.lo[0], dy = scene.hi[1] - scene.lo[1], dz = scene.hi[2] - scene.lo[2];
  out.diag = nt ? std::sqrt(dx * dx + dy * dy + dz * dz) : 0.f;
  // Child boxes are inflated before quantisation so that fp32 slab tests can never cull a triangle the exact
  // test accepts: slab rounding moves an entry/exit point by < 2e-7 * diag, the inflation is 20 times that.
  // Quantisation then only rounds outwards.
  const float pad = 4e-6f * out.diag;
  out.nodes.clear();
  out.tris.clear();
  out.depth = 0;
  out.sah_cost = 0.f;
  if (!nt) {
    NodeC root;
    std::memset(&root, 0, sizeof(root));
    for (int a = 0; a < 3; ++a) {
      root.e[a] = 127;
      for (int s = 0; s < 8; ++s) { root.qlo[a][s] = 255; root.qhi[a][s] = 0; }
    }
    out.nodes.push_back(root);
    out.depth = 1;
    return;
  }
  Builder b(tb, cen);
  b.leaf_max = g_optimal_collapse ? 1u : (uint32_t)kMaxLeafTris;
  b.build(0, nr);
  const std::vector<Node2>& n2 = b.nodes;

  auto emit_tri = [&](uint32_t id) {
    const float* a = &verts[3 * idx[3 * id]];
    const float* bb = &verts[3 * idx[3 * id + 1]];
    const float* c = &verts[3 * idx[3 * id + 2]];
    TriPacked tp;
    for (int x = 0; x < 3; ++x) { tp.v0[x] = a[x]; tp.e1[x] = bb[x] - a[x]; tp.e2[x] = c[x] - a[x]; }
    tp.id = id; tp.mat = tri_mat[id]; tp.pad = 0;
    out.tris.push_back(tp);
  };
  out.tris.reserve(nr);

  // ---- which BVH2 subtrees become the children of one BVH8 node
  // g_optimal_collapse: the cost-optimal cut (dynamic programme over the BVH2, restated from section 3.1 of Ylitie, Karras
  // and Laine 2017): cost[n][i] = least SAH cost of representing the subtree of n by at most i + 1 roots (leaves of at most
  // kMaxLeafTris references, or BVH8 nodes), area(n) * kCostNode per node and area * refs * kCostTri per leaf.  The BVH2 is
  // built down to single references, so the programme also decides what a leaf is.  Otherwise: greedy, open the child of
  // largest area until there are eight.  Measured on configs[3]: profiles/r02b_tuning.md (BVH collapse table).
  constexpr int kW = 8;
  const size_t nn2 = n2.size();
  std::vector<float> cost;          // [n * 7 + i], i = 0..6: at most i + 1 roots
  std::vector<uint8_t> pick;        // [n * 8 + i]: i < 7: roots given to the left child when n is distributed over i + 1 roots
                                    //   (0 = not distributed: same as i - 1, or for i = 0 one root: see kind); [n * 8 + 7]: for the 8-way distribution of a node
  std::vector<uint8_t> kind;        // [n]: 1 = a single root at n is a leaf, 0 = a BVH8 node
  if (g_optimal_collapse) {
    cost.assign(nn2 * 7, 0.f); pick.assign(nn2 * 8, 0); kind.assign(nn2, 0);
    for (size_t n = nn2; n-- > 0;) {   // children have larger indices than their parent (pre-order)
      const Node2& N = n2[n];
      const float A = N.box.area();
      float* c = &cost[n * 7];
      if (N.count) {                   // BVH2 leaf: one reference
        for (int i = 0; i < 7; ++i) c[i] = A * kCostTri * (float)N.refs;
        kind[n] = 1;
        continue;
      }
      const float* cl = &cost[(size_t)N.left * 7];
      const float* cr = &cost[(size_t)N.right * 7];
      auto distribute = [&](int roots, uint8_t& k_best) {   // roots >= 2 split between the two children
        float best = FLT_MAX;
        for (int k = 1; k < roots; ++k) {
          if (k > 7 || roots - k > 7) continue;
          const float v = cl[k - 1] + cr[roots - k - 1];
          if (v < best) { best = v; k_best = (uint8_t)k; }
        }
        return best;
      };
      uint8_t k8 = 1;
      const float as_node = A * kCostNode + distribute(kW, k8);
      pick[n * 8 + 7] = k8;
      const float as_leaf = N.refs <= (uint32_t)kMaxLeafTris ? A * kCostTri * (float)N.refs : FLT_MAX;
      kind[n] = as_leaf <= as_node ? 1 : 0;
      c[0] = std::min(as_leaf, as_node);
      for (int i = 1; i < 7; ++i) {
        uint8_t k = 0;
        const float d = distribute(i + 1, k);
        if (d < c[i - 1]) { c[i] = d; pick[n * 8 + i] = k; } else { c[i] = c[i - 1]; pick[n * 8 + i] = 0; }
      }
    }
  }
  // roots of the subtree of n when it may use `roots` of them
  struct Expand {
    const std::vector<Node2>& n2; const std::vector<uint8_t>& pick;
    void run(uint32_t n, int roots, uint32_t* out, int& cnt) const {
      while (roots > 1 && pick[(size_t)n * 8 + roots - 1] == 0) --roots;   // fewer roots were as good
      if (roots == 1 || n2[n].count) { out[cnt++] = n; return; }
      const int k = pick[(size_t)n * 8 + roots - 1];
      run(n2[n].left, k, out, cnt);
      run(n2[n].right, roots - k, out, cnt);
    }
  };
  auto is_leaf = [&](uint32_t n) { return g_optimal_collapse ? kind[n] != 0 : n2[n].count != 0; };

  // collapse to BVH8, breadth-first; a node's index is its position in the queue order
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
    if (g_optimal_collapse) {
      if (it.n2 == 0 && n2[0].refs <= (uint32_t)kMaxLeafTris) { kind[0] = 1; kids[nk++] = 0; }   // the whole scene is one leaf
      else {
        const int k = pick[(size_t)it.n2 * 8 + 7];
        const Expand ex{n2, pick};
        ex.run(n2[it.n2].left, k, kids, nk);
        ex.run(n2[it.n2].right, kW - k, kids, nk);
      }
    } else {
      if (n2[it.n2].count) kids[nk++] = it.n2;  // the root is itself a leaf
      else { kids[nk++] = n2[it.n2].left; kids[nk++] = n2[it.n2].right; }
      for (;;) {  // open the internal child with the largest area until 8 children
        if (nk == 8) break;
        int pick_i = -1;
        float pa = -1.f;
        for (int i = 0; i < nk; ++i)
          if (!n2[kids[i]].count && n2[kids[i]].box.area() > pa) { pa = n2[kids[i]].box.area(); pick_i = i; }
        if (pick_i < 0) break;
        const uint32_t p = kids[pick_i];
        kids[pick_i] = n2[p].left;
        kids[nk++] = n2[p].right;
      }
    }
    int slot_of[8];
    assign_slots(n2, kids, nk, slot_of);
    int kid_in_slot[8];
    for (int s = 0; s < 8; ++s) kid_in_slot[s] = -1;
    for (int i = 0; i < nk; ++i) kid_in_slot[slot_of[i]] = i;

    NodeC node;
    std::memset(&node, 0, sizeof(node));
    node.child_base = next_index;
    node.tri_base = (uint32_t)out.tris.size();
    // padded child boxes and the node grid
    Box cb[8], nb;
    for (int s = 0; s < 8; ++s) {
      if (kid_in_slot[s] < 0) continue;
      const Node2& c = n2[kids[kid_in_slot[s]]];
      for (int a = 0; a < 3; ++a) { cb[s].lo[a] = c.box.lo[a] - pad; cb[s].hi[a] = c.box.hi[a] + pad; }
      nb.grow(cb[s]);
    }
    for (int a = 0; a < 3; ++a) {
      node.p[a] = nb.lo[a];
      const double p = (double)nb.lo[a], ext = (double)nb.hi[a] - p;
      int e = ext > 0.0 ? (int)std::ceil(std::log2(ext / 255.0)) : -120;
      e = std::max(e, -120);
      for (;;) {
        const double cell = std::ldexp(1.0, e);
        bool ok = true;
        for (int s = 0; s < 8 && ok; ++s) {
          if (kid_in_slot[s] < 0) { node.qlo[a][s] = 255; node.qhi[a][s] = 0; continue; }  // inverted: never hit
          // outward rounding with 0.01 cell of slack for the kernel's plane arithmetic (dr_traverse.cuh node_hits)
          double ql = std::floor(((double)cb[s].lo[a] - p) / cell - 0.01);
          while (ql > 0.0 && p + (ql + 0.01) * cell > (double)cb[s].lo[a]) ql -= 1.0;
          double qh = std::ceil(((double)cb[s].hi[a] - p) / cell + 0.01);
          while (p + (qh - 0.01) * cell < (double)cb[s].hi[a]) qh += 1.0;
          if (ql < 0.0) ql = 0.0;
          if (qh > 255.0) { ok = false; break; }
          node.qlo[a][s] = (uint8_t)ql;
          node.qhi[a][s] = (uint8_t)qh;
        }
        if (ok) break;
        ++e;
      }
      node.e[a] = (uint8_t)(e + 127);
    }
    for (int s = 0; s < 8; ++s) {
      if (kid_in_slot[s] < 0) continue;
      const Node2& c = n2[kids[kid_in_slot[s]]];
      if (is_leaf(kids[kid_in_slot[s]])) {
        node.trimask |= ((1u << c.refs) - 1u) << (3 * s);
        for (uint32_t k = 0; k < c.refs; ++k) emit_tri(refs[b.order[c.first + k]].tri);
        sah += (double)c.box.area() / root_area * c.refs;
      } else {
        node.imask |= (uint8_t)(1u << s);
        ++next_index;
        q.push({kids[kid_in_slot[s]], it.depth + 1});
        sah += (double)c.box.area() / root_area;
      }
    }
    node.imask32 = node.imask;
    out.nodes.push_back(node);
  }
  out.sah_cost = (float)sah;
}

}  // namespace dr
