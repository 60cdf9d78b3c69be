// Internal types shared by the host-side scene builder and the kernels.
#pragma once
#include <cstddef>
#include <cstdint>
#include <vector>

namespace dr {

constexpr int kMaxPathLen = 16;        // L <= 16, d = 2L <= 32 (BASELINE.json configs[3])
constexpr int kMaxPlanes = 8;          // d / 4 float4 planes
constexpr uint32_t kLeafBit = 0x80000000u;
constexpr uint32_t kEmptyChild = 0xFFFFFFFFu;
constexpr int kSmemNodes = 73;         // root + 8 + 64: the top three BVH8 levels staged in shared memory
constexpr int kMaxMix = 16;

// BVH8 node, 256 bytes, child boxes as structure-of-arrays so a lane reads them as float4 pairs.
// child[i]: kEmptyChild, or internal node index, or kLeafBit | (count-1) << 27 | first triangle (leaf order).
struct alignas(256) Node8 {
  float lo[3][8];
  float hi[3][8];
  uint32_t child[8];
  uint32_t pad[8];
};
static_assert(sizeof(Node8) == 256, "Node8 must be 256 bytes");

// Triangle in leaf order, 48 bytes: three float4.
//   q0 = (v0.xyz, bits(original triangle id)), q1 = (e1.xyz, bits(material id)), q2 = (e2.xyz, 0)
struct TriPacked {
  float v0[3]; uint32_t id;
  float e1[3]; uint32_t mat;
  float e2[3]; uint32_t pad;
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
  std::vector<Node8> nodes;         // breadth-first order: node 0 = root, top levels first
  std::vector<TriPacked> tris;      // leaf order
  uint32_t depth = 0;
  float sah_cost = 0.f;
  float diag = 0.f;
};

// Binned-SAH BVH2 -> BVH8 collapse (host).  verts: 3*nv floats, idx: 3*nt, tri_mat: nt.
void build_bvh8(const float* verts, uint32_t nv, const uint32_t* idx, uint32_t nt, const uint32_t* tri_mat, BuiltBvh& out);

}  // namespace dr
