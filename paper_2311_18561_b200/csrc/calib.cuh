// calib.cuh -- measurement hook: the FP32 / issue-slot peak of THIS device, measured, for the roofline of the
// ALU-bound blend ("verify SM count with cudaGetDeviceProperties and calibrate with an FFMA
// microbenchmark on the box"). Not on the render path.
//
// Every thread runs 8 independent dependency chains (a chain's next instruction issues 4+ cycles after the
// previous one; 8 warps per scheduler x 8 chains cover that many times over), 64 or 128 instructions per
// loop trip, so loop overhead is 2-3 %:
//   mode 0: FFMA only, three register operands (the form the blend's inner loop uses)
//   mode 1: FFMA and LOP3 alternating -- the FMA pipe and the ALU pipe side by side, the mix an issue-bound
//           kernel like the blend (FFMA/FMUL/FADD + FMNMX/FSETP/SEL/LOP3) presents to the scheduler
//   mode 2: FFMA2 (fma.rn.f32x2, sm_100+): two fp32 FMAs per lane per instruction
#pragma once

#include "common.cuh"

namespace pvg {

constexpr int CALIB_THREADS = 256;
constexpr int CALIB_CHAINS = 8;
constexpr int CALIB_UNROLL = 8;

template <int MODE>
__global__ void __launch_bounds__(CALIB_THREADS)
calib_kernel(float* __restrict__ sink, int trips, float a, float b, uint32_t c, uint32_t d) {
  float x[CALIB_CHAINS];
  uint32_t y[CALIB_CHAINS];
  unsigned long long z[CALIB_CHAINS];
#pragma unroll
  for (int k = 0; k < CALIB_CHAINS; ++k) {
    x[k] = (float)(threadIdx.x + k) * 1e-3f;
    y[k] = threadIdx.x * 2654435761u + k;
    z[k] = ((unsigned long long)__float_as_uint(x[k]) << 32) | __float_as_uint(x[k] + 1.0f);
  }
  const unsigned long long a2 = ((unsigned long long)__float_as_uint(a) << 32) | __float_as_uint(a);
  const unsigned long long b2 = ((unsigned long long)__float_as_uint(b) << 32) | __float_as_uint(b);
#pragma unroll 1
  for (int t = 0; t < trips; ++t) {
#pragma unroll
    for (int u = 0; u < CALIB_UNROLL; ++u) {
#pragma unroll
      for (int k = 0; k < CALIB_CHAINS; ++k) {
        if (MODE == 2) {
          asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(z[k]) : "l"(a2), "l"(b2));
        } else {
          asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(x[k]) : "f"(a), "f"(b));
          if (MODE == 1) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(y[k]) : "r"(c), "r"(d));
        }
      }
    }
  }
  float s = 0.f;
  uint32_t q = 0;
#pragma unroll
  for (int k = 0; k < CALIB_CHAINS; ++k) {
    s += x[k] + __uint_as_float((uint32_t)z[k]) + __uint_as_float((uint32_t)(z[k] >> 32));
    q ^= y[k];
  }
  if (s == 1.2345e-30f && q == 0x12345u) sink[blockIdx.x * CALIB_THREADS + threadIdx.x] = s;   // never true: keeps the chains
}

// thread-level instructions one launch executes (a packed FFMA2 counts once: it is one issue slot)
__host__ inline double calib_instructions(int mode, unsigned grid, int trips) {
  const double per_trip = (double)CALIB_UNROLL * CALIB_CHAINS * (mode == 1 ? 2.0 : 1.0);
  return (double)grid * CALIB_THREADS * (double)trips * per_trip;
}

}  // namespace pvg
