// Hardware probes behind thc_probe (include/thc.h): the measured ceilings that the FP64 kernels of this library are
// judged against.  MEASURED_PEAKS.json has no FP64 entry, so the library measures its own:
//   * issue rate of the FP64 tensor instruction (mma.sync.m8n8k4.f64, SASS DMMA.8x8x4) -- roof of the GEMM chains,
//   * issue rate of DFMA -- roof of Alg.6 line 11,
//   * both interleaved in one warp -- shows whether they share a pipe,
//   * shared memory -> register bandwidth by access width -- the operand roof of the line-11 register tile.
// Every probe is a persistent grid of one 256-thread CTA per SM running a register-resident loop; the host times it with
// CUDA events.  Nothing here is on the product path.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "thc_gemm.cuh"

namespace thc {

constexpr int PROBE_THREADS = 256, PROBE_UNROLL = 8;

// mode 0: DMMA only, 1: DFMA only, 2: interleaved (PROBE_UNROLL of each per iteration)
template <int MODE>
__global__ void __launch_bounds__(PROBE_THREADS) probe_fp64_kernel(double* sink, int iters, double seed) {
  double acc[PROBE_UNROLL][2], f[PROBE_UNROLL];
#pragma unroll
  for (int k = 0; k < PROBE_UNROLL; k++) { acc[k][0] = acc[k][1] = 0.0; f[k] = seed + k; }
  const double a = seed * 1e-3 + threadIdx.x * 1e-9, b = 1.0 - seed * 1e-6;
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int k = 0; k < PROBE_UNROLL; k++) {
      if (MODE != 1) dmma884(acc[k][0], acc[k][1], a, b);
      if (MODE != 0) f[k] = fma(f[k], b, a);
    }
  }
  double s = 0.0;
#pragma unroll
  for (int k = 0; k < PROBE_UNROLL; k++) s += acc[k][0] + acc[k][1] + f[k];
  if (s == 123.456) sink[0] = s;          // never true: keeps the loop alive
}

// WIDTH = 4, 8 or 16 bytes per lane per load; lanes read consecutive addresses (conflict-free).  Eight independent load
// chains per thread: the address of a load depends on the value the previous load of its chain returned (through
// `mask`, which is 0 at run time but unknown to the compiler), so no load can be merged, hoisted or dropped, while
// 8 chains x 8 warps keep far more loads in flight than the ~30-cycle latency needs.
template <int WIDTH>
__global__ void __launch_bounds__(PROBE_THREADS) probe_lds_kernel(unsigned* sink, int iters, unsigned mask) {
  __shared__ __align__(16) unsigned buf[PROBE_THREADS * 4 * 2];
  for (int i = threadIdx.x; i < PROBE_THREADS * 8; i += PROBE_THREADS) buf[i] = i * 2654435761u;
  __syncthreads();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const unsigned base = (unsigned)__cvta_generic_to_shared(buf + warp * 32 * (WIDTH / 4) + lane * (WIDTH / 4));
  unsigned x[8];
#pragma unroll
  for (int k = 0; k < 8; k++) x[k] = k;
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int k = 0; k < 8; k++) {
      const unsigned addr = base + (((x[k] & mask) + k) & 1) * (PROBE_THREADS * 16);
      if (WIDTH == 4) {
        unsigned v;
        asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
        x[k] ^= v;
      } else if (WIDTH == 8) {
        uint2 v;
        asm volatile("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr) : "memory");
        x[k] ^= v.x ^ v.y;
      } else {
        uint4 v;
        asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr) : "memory");
        x[k] ^= v.x ^ v.y ^ v.z ^ v.w;
      }
    }
  }
  unsigned r = 0;
#pragma unroll
  for (int k = 0; k < 8; k++) r ^= x[k];
  if (r == 0x12345678u) sink[0] = r;
}

}  // namespace thc
