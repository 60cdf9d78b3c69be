// Internal types shared by the host-side scene builder and the kernels.
#pragma once
#include <cstddef>
#include <cstdint>
#include <vector>

namespace dr {

constexpr int kMaxPathLen = 16;        // L <= 16: d = 2L <= 32 (BASELINE.json configs[3]), or d = 4L <= 64 with next-event estimation
                                       // (Q21); the state is stored in d / 4 float4 planes (DevScene::planes)
constexpr int kMaxMix = 16;
constexpr int kMaxLeafTris = 3;        // triangles per leaf (three bits per slot in the node's triangle mask)
constexpr int kMaxBvhDepth = 30;       // upper bound; what the traversal stacks in shared memory allow is checked by dr_scene_create

// BVH8 node, 80 bytes = five 16-byte words.  Child boxes are quantised to 8 bits per plane on a per-node
// grid (origin p, per-axis power-of-two cell 2^(e-127)), rounded outwards, so a node costs five 128-bit loads.
//   w0 = (p.x, p.y, p.z, e_x | e_y << 8 | e_z << 16 | imask << 24)      imask: bit s = slot s is an internal node
//   w1 = (child_base, tri_base, trimask, imask)      imask again as a word: every loaded register is read (see TriPacked)
//   w2 = (qlo_x[0..3], qlo_x[4..7], qlo_y[0..3], qlo_y[4..7])
//   w3 = (qlo_z[0..3], qlo_z[4..7], qhi_x[0..3], qhi_x[4..7])
//   w4 = (qhi_y[0..3], qhi_y[4..7], qhi_z[0..3], qhi_z[4..7])
// trimask: bit 3 s + k is set iff slot s is a leaf with more than k triangles (k < 3).  The triangles of a node are
// stored contiguously from tri_base in the order of their bits: the triangle of bit b is
// tri_base + popcount(trimask & ((1 << b) - 1)).  Fixed bit positions let the node test build its work mask with one
// select per child (dr_traverse.cuh node_hits); an empty slot has inverted boxes and no bit in either mask.
// Internal children of a node are stored contiguously from child_base in slot order: the child in slot s is
// node child_base + popcount(imask & ((1 << s) - 1)).  Slots are assigned so that children lie towards corner
// (s&4 ? +x : -x, s&2 ? +y : -y, s&1 ? +z : -z) of the node: visiting slots in the order of descending
// (s ^ octinv), octinv = (d.x >= 0 ? 4 : 0) | (d.y >= 0 ? 2 : 0) | (d.z >= 0 ? 1 : 0), is roughly front to back.
struct alignas(16) NodeC {
  float p[3];
  uint8_t e[3];
  uint8_t imask;
  uint32_t child_base, tri_base;
  uint32_t trimask, imask32;
  uint8_t qlo[3][8];
  uint8_t qhi[3][8];
};
static_assert(sizeof(NodeC) == 80, "NodeC must be 80 bytes");

// Triangle in leaf order, 48 bytes = three 16-byte words:
//   t0 = (v0.x, v0.y, v0.z, e1.x), t1 = (e1.y, e1.z, e2.x, e2.y), t2 = (e2.z, bits(original id), bits(material id), 0)
// The traversal loads t0, t1 and the first half of t2 (40 bytes), so that every register a load writes is read by
// the triangle test (a loaded-but-unread register is free for reuse while the load is still in flight, which made
// the next write to it wait for the whole load: profiles/r01f_k_trace_full.md, step r01e).
struct TriPacked {
  float v0[3];
  float e1[3];
  float e2[3];
  uint32_t id, mat, pad;
};
static_assert(sizeof(TriPacked) == 48, "TriPacked must be 48 bytes");

// Material, 48 bytes: three float4.  q0 = (bits(kind), a0, a1, a2), q1 = (ior, alpha, Le0, Le1), q2 = (Le2, 0, 0, 0)
struct MatPacked {
  uint32_t kind; float a[3];
  float ior, alpha, le0, le1;
  float le2, pad[3];
};
static_assert(sizeof(MatPacked) == 48, "MatPacked must be 48 bytes");

struct BuiltBvh {
  std::vector<NodeC> nodes;         // breadth-first order: node 0 = root, top levels first
  std::vector<TriPacked> tris;      // leaf order (the leaves of one node are contiguous)
  uint32_t depth = 0;               // levels of BVH8 nodes
  float sah_cost = 0.f;
  float diag = 0.f;
};

// Binned-SAH BVH2 -> BVH8 collapse -> slot assignment -> quantisation (host).  verts: 3*nv floats, idx: 3*nt, tri_mat: nt.
void set_split_budget(double extra_refs_per_triangle);  // tuning hook (default DR_SPLIT_BUDGET)
void set_collapse(bool optimal, float cost_node, float cost_tri);   // tuning hook: BVH2 -> BVH8 collapse (dr_bvh.cpp)
void build_bvh8(const float* verts, uint32_t nv, const uint32_t* idx, uint32_t nt, const uint32_t* tri_mat, BuiltBvh& out);

}  // namespace dr
