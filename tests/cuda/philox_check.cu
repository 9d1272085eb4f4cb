// Test-only helper (never loaded by the product): evaluates (a) the product's Philox4x32-10 device function
// and (b) cuRAND's curand_Philox4x32_10 from the CUDA toolkit header on the same (counter, key) pairs, so that
// tests/test_gpu_parity.py can compare both with the oracle and the big-integer writing.  DESIGN.md "C3".
#include <cuda_runtime.h>
#include <curand_kernel.h>
#include <curand_philox4x32_x.h>
#include <stdint.h>

#include "../../paper_2006_00561_b200/csrc/pa_common.cuh"

__global__ void k_both(const uint32_t* ctr, const uint32_t* key, uint32_t* out_lib, uint32_t* out_curand, int n) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  pa::PhiloxKey pk;
  uint32_t k0 = key[2 * i], k1 = key[2 * i + 1];
  for (int r = 0; r < 10; ++r) {
    pk.k0[r] = k0;
    pk.k1[r] = k1;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  const uint4 a = pa::philox4x32_10(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3], pk);
  out_lib[4 * i] = a.x; out_lib[4 * i + 1] = a.y; out_lib[4 * i + 2] = a.z; out_lib[4 * i + 3] = a.w;
  const uint4 b = curand_Philox4x32_10(make_uint4(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3]),
                                       make_uint2(key[2 * i], key[2 * i + 1]));
  out_curand[4 * i] = b.x; out_curand[4 * i + 1] = b.y; out_curand[4 * i + 2] = b.z; out_curand[4 * i + 3] = b.w;
}

// all pointers DEVICE; returns cudaError_t as int
extern "C" int philox_check(const uint32_t* ctr, const uint32_t* key, uint32_t* out_lib, uint32_t* out_curand, int n) {
  k_both<<<(n + 255) / 256, 256>>>(ctr, key, out_lib, out_curand, n);
  return (int)cudaDeviceSynchronize();
}
