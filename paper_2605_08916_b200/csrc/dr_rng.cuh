// Counter-based Philox4x32-10 for the chain kernels (row a1).  The paper keeps a Philox state per chain
// (PAPER.md L480, L500); here the generator is stateless: key = (seed lo, seed hi), counter =
// (chain, iteration, slot, purpose | epoch << 8) (Q14), so no RNG state is stored or moved.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace dr {

enum Purpose : uint32_t { P_REGEN_U = 0, P_PROP_N = 1, P_DECIDE = 2, P_LARGE_U = 3 };

__device__ __forceinline__ uint4 philox4x32_10(uint2 key, uint4 c) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
    c = make_uint4(hi1 ^ c.y ^ key.x, lo1, hi0 ^ c.w ^ key.y, lo0);
    key.x += 0x9E3779B9u;
    key.y += 0xBB67AE85u;
  }
  return c;
}

__device__ __forceinline__ uint4 stream_block(uint64_t seed, uint32_t chain, uint32_t iteration, uint32_t slot,
                                              uint32_t purpose, uint32_t epoch) {
  return philox4x32_10(make_uint2((uint32_t)seed, (uint32_t)(seed >> 32)),
                       make_uint4(chain, iteration, slot, purpose | (epoch << 8)));
}

// u in [0,1) and u in (0,1] from the top 24 bits (exact in fp32).
__device__ __forceinline__ float u01_co(uint32_t w) { return (float)(w >> 8) * 5.9604644775390625e-8f; }
__device__ __forceinline__ float u01_oc(uint32_t w) { return (float)((w >> 8) + 1u) * 5.9604644775390625e-8f; }

__device__ __forceinline__ float4 uniforms4(uint4 w) { return make_float4(u01_co(w.x), u01_co(w.y), u01_co(w.z), u01_co(w.w)); }

// Box-Muller: (wa, wb) -> N(0, I_2), the xi of Alg. 4 line 3.  Accurate logf / sincosf.
__device__ __forceinline__ float2 box_muller(uint32_t wa, uint32_t wb) {
  const float r = sqrtf(-2.0f * logf(u01_oc(wa)));
  float s, c;
  sincosf(6.283185307179586f * u01_co(wb), &s, &c);
  return make_float2(r * c, r * s);
}

__device__ __forceinline__ float4 normals4(uint4 w) {
  const float2 a = box_muller(w.x, w.y), b = box_muller(w.z, w.w);
  return make_float4(a.x, a.y, b.x, b.y);
}

}  // namespace dr
