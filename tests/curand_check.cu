// TEST INFRASTRUCTURE -- third leg of the Philox4x32-10 check (SURVEY.md 8c pins): cuRAND's own device function on the
// same (key, counter) pairs.  Built by tests/test_gpu_parity.py with nvcc on the GPU box; shares nothing with csrc/ or oracle/.
#include <cstdint>
#include <curand_kernel.h>
#include <curand_philox4x32_x.h>

__global__ void k_curand_philox(uint2 key, const uint32_t* ctr, uint32_t n, uint32_t* out) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint4 r = curand_Philox4x32_10(make_uint4(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3]), key);
  out[4 * i] = r.x; out[4 * i + 1] = r.y; out[4 * i + 2] = r.z; out[4 * i + 3] = r.w;
}

// device pointers; returns the cudaError_t of the launch + synchronisation
extern "C" int curand_philox_blocks(uint64_t seed, const uint32_t* dev_ctr, uint32_t n, uint32_t* dev_out) {
  k_curand_philox<<<(n + 255) / 256, 256>>>(make_uint2((uint32_t)seed, (uint32_t)(seed >> 32)), dev_ctr, n, dev_out);
  return (int)cudaDeviceSynchronize();
}
