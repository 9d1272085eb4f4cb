// pipe_probe.cu -- measurement tool behind the roofline of the sweep kernel (profiles/r2_pipe_probe.md).
// Not part of the library.  How many SMSP cycles does one warp need for a mix of IMAD.WIDE.U32 (FMA-heavy pipe; Philox's
// 32 x 32 -> 64 multiplies) and LOP3 (ALU pipe), with the sweep kernel's occupancy (128-thread blocks, 4 per SM = 4 warps
// per SMSP) and 8 independent chains per thread?  Timed with CUDA events over 20 000 iterations; cycles at 1965 MHz.
//   nvcc -O3 -gencode arch=compute_100a,code=sm_100a -o gpurun_out/pipe_probe paper_2006_00561_b200/csrc/pipe_probe.cu
#include <cstdio>
#include <cuda_runtime.h>
#include <stdint.h>
constexpr int NCH = 8;  // independent chains per thread
// NM = IMAD.WIDE per chain and iteration (0 or 2), NL = extra LOP3 per chain and iteration beyond the 2 that consume the
// products (0, 2, 4); NM = 0: LOP3 only (NL + 2 per chain)
template <int NM, int NL>
__global__ void __launch_bounds__(128, 4) k(uint32_t* out, int iters, uint32_t seed) {
  uint32_t a[NCH], b[NCH], c[NCH], d[NCH];
  for (int i = 0; i < NCH; ++i) { a[i] = seed + threadIdx.x * 7 + i; b[i] = a[i] * 3; c[i] = a[i] ^ 0x55; d[i] = a[i] + 9; }
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < NCH; ++i) {
      if (NM == 2) {
        uint32_t lo, hi, lo2, hi2;
        asm volatile("{.reg .u64 t; mul.wide.u32 t, %2, 0xD2511F53; mov.b64 {%0,%1}, t;}" : "=r"(lo), "=r"(hi) : "r"(a[i]));
        asm volatile("{.reg .u64 t; mul.wide.u32 t, %2, 0xCD9E8D57; mov.b64 {%0,%1}, t;}" : "=r"(lo2), "=r"(hi2) : "r"(b[i]));
        asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(a[i]) : "r"(hi2), "r"(lo), "r"(c[i]));
        asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(b[i]) : "r"(hi), "r"(lo2), "r"(d[i]));
      } else {
        asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a[i]) : "r"(c[i]), "r"(d[i]));
        asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(b[i]) : "r"(c[i]), "r"(d[i]));
      }
      if (NL >= 2) {
        asm volatile("lop3.b32 %0, %0, %1, %2, 0xca;" : "+r"(c[i]) : "r"(a[i]), "r"(d[i]));
        asm volatile("lop3.b32 %0, %0, %1, %2, 0x90;" : "+r"(d[i]) : "r"(b[i]), "r"(c[i]));
      }
      if (NL >= 4) {
        asm volatile("lop3.b32 %0, %0, %1, %2, 0xca;" : "+r"(c[i]) : "r"(b[i]), "r"(d[i]));
        asm volatile("lop3.b32 %0, %0, %1, %2, 0x90;" : "+r"(d[i]) : "r"(a[i]), "r"(c[i]));
      }
    }
  }
  uint32_t s = 0;
  for (int i = 0; i < NCH; ++i) s ^= a[i] ^ b[i] ^ c[i] ^ d[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
template <int NM, int NL>
void run() {
  uint32_t* out;
  cudaMalloc(&out, 148 * 4 * 128 * 4);
  const int iters = 20000;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  k<NM, NL><<<148 * 4, 128>>>(out, iters, 1);  // warm-up
  cudaEventRecord(e0);
  k<NM, NL><<<148 * 4, 128>>>(out, iters, 1);
  cudaEventRecord(e1);
  cudaEventSynchronize(e1);
  float ms;
  cudaEventElapsedTime(&ms, e0, e1);
  const int nm = NM * NCH, nl = (2 + NL) * NCH;
  const double cyc = ms * 1e-3 * 1.965e9 / iters / 4;  // 4 warps share an SMSP
  printf("| %2d IMAD.WIDE.U32 + %2d LOP3 | %6.1f | %5.2f | %3d / %3d |\n", nm, nl, cyc, cyc / (nm + nl), 4 * nm > 2 * nl ? 4 * nm : 2 * nl,
         2 * (nm + nl));
  cudaFree(out);
}
int main() {
  printf("| mix per warp and iteration | SMSP cycles per warp-iteration | cycles per instruction | max(4 IMADW, 2 LOP3) / 2 (IMADW + LOP3) |\n|---|---|---|---|\n");
  run<0, 4>();  // 48 LOP3
  run<2, 0>();  // 16 + 16
  run<2, 2>();  // 16 + 32
  run<2, 4>();  // 16 + 48
  run<0, 0>();  // 16 LOP3
  return 0;
}
