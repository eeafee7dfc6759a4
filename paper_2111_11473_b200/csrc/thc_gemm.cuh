// FP64 DMMA GEMM for sm_100a: the one kernel every GEMM chain of the THC-RR-CCSD residual runs on.
//
//   C_b[m][n] = alpha * ( sum_{kb < kbatch} sum_{k < K} A_{b,kb}(m,k) * B_{b,kb}(n,k) ) (.* aux_b[m][n]) + beta * C_b[m][n]
//
// A(m,k) = A[m*lda + k] ("K-major") or A[k*lda + m] ("M-major"); likewise B(n,k).  `kbatch` is a second,
// strided K loop (sum over Cholesky vectors of D^L C^L^T, Alg.1 line 15 l.524); `splits` cuts the
// combined K range over grid.z and writes partial tiles that reduce_splits_kernel adds up in a fixed order.
//
// Tensor-core path: on sm_100a every FP64 mma.sync shape is issued as DMMA.8x8x4 (checked with cuobjdump),
// so the kernel uses m8n8k4 directly.  Fragment ownership (lane = 4*g + t):
//   A: (row g, k t)   B: (k t, col g)   C: (row g, cols 2t, 2t+1).
// Within each group of 8 k the two k4 steps take k = 2t + h (h = 0, 1): a K-major operand is stored in
// shared memory as [k/8][row][8] so that one conflict-free 16-byte load gives a lane both steps' values; an
// M/N-major operand is stored as [k][rows + 2] (pitch = 16 B mod 128 B) and read with conflict-free 8-byte loads.
// Global -> shared copies are cp.async (16 B when pointers/strides allow, else 8 B) in a STAGES-deep ring.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace thc {

struct GemmParams {
  const double* A; const double* B; double* C; const double* aux;
  int M, N, K;
  long long lda, ldb, ldc, ldaux;
  int batch; long long sAb, sBb, sCb, sAuxb;
  int kbatch; long long sAk, sBk;
  int splits; long long sCs;      // split-K: partial tile stride (C then points at the partial buffer)
  double alpha, beta;
};

__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem, int src_bytes) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(s), "l"(gmem), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async8(void* smem, const void* gmem, int src_bytes) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(s), "l"(gmem), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N)); }

// Copy one BK-deep slab of an operand tile (ROWS rows starting at row0 of an operand with `nrows` rows) into smem.
template <int ROWS, int BK, int NTHREADS, bool KMAJOR, bool AL16>
__device__ __forceinline__ void load_tile(double* s, const double* __restrict__ g, long long ld, int row0, int nrows,
                                          int k0, int K, int tid) {
  if (KMAJOR) {
    // smem [BK/8][ROWS][8]; global row r: g[r*ld + k]
    constexpr int CHUNKS = ROWS * BK / 2;
    for (int c = tid; c < CHUNKS; c += NTHREADS) {
      int kb8 = c / (ROWS * 4), rem = c % (ROWS * 4), r = rem / 4, cc = rem % 4;
      int k = k0 + kb8 * 8 + cc * 2;
      int row = row0 + r;
      double* dst = s + (kb8 * ROWS + r) * 8 + cc * 2;
      bool rok = row < nrows;
      const double* src = g + (rok ? (long long)row * ld : 0) + (k < K ? k : 0);
      int nb = rok ? max(0, min(2, K - k)) * 8 : 0;
      if (AL16) {
        cp_async16(dst, src, nb);
      } else {
        cp_async8(dst, src, nb >= 8 ? 8 : 0);
        cp_async8(dst + 1, nb >= 16 ? src + 1 : src, nb >= 16 ? 8 : 0);
      }
    }
  } else {
    // smem [BK][ROWS+2]; global: g[k*ld + r]
    constexpr int PITCH = ROWS + 2;
    constexpr int CHUNKS = BK * ROWS / 2;
    for (int c = tid; c < CHUNKS; c += NTHREADS) {
      int kk = c / (ROWS / 2), cc = c % (ROWS / 2);
      int k = k0 + kk, row = row0 + cc * 2;
      double* dst = s + kk * PITCH + cc * 2;
      bool kok = k < K;
      const double* src = g + (kok ? (long long)k * ld : 0) + (row < nrows ? row : 0);
      int nb = kok ? max(0, min(2, nrows - row)) * 8 : 0;
      if (AL16) {
        cp_async16(dst, src, nb);
      } else {
        cp_async8(dst, src, nb >= 8 ? 8 : 0);
        cp_async8(dst + 1, nb >= 16 ? src + 1 : src, nb >= 16 ? 8 : 0);
      }
    }
  }
}

template <int BM, int BN, int BK, int WM, int WN, int STAGES, bool AKM, bool BKM, bool AL16>
__global__ void __launch_bounds__(WM* WN * 32) dgemm_kernel(const GemmParams p) {
  constexpr int NTHREADS = WM * WN * 32;
  constexpr int WTM = BM / WM, WTN = BN / WN, MT = WTM / 8, NT = WTN / 8;
  constexpr int A_STAGE = AKM ? BM * BK : BK * (BM + 2);
  constexpr int B_STAGE = BKM ? BN * BK : BK * (BN + 2);
  extern __shared__ __align__(16) double smem[];
  double* sA = smem;
  double* sB = smem + STAGES * A_STAGE;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, g = lane >> 2, t = lane & 3;
  const int wm = warp / WN, wn = warp % WN;
  const int tiles_n = (p.N + BN - 1) / BN;
  const int tile_m = blockIdx.x / tiles_n, tile_n = blockIdx.x % tiles_n;
  const int split = blockIdx.z % p.splits, b = blockIdx.z / p.splits;
  const int m0 = tile_m * BM, n0 = tile_n * BN;
  const double* Ab = p.A + (long long)b * p.sAb;
  const double* Bb = p.B + (long long)b * p.sBb;
  const int ktiles = (p.K + BK - 1) / BK;
  const int total_it = p.kbatch * ktiles;
  const int it_begin = (int)((long long)total_it * split / p.splits);
  const int it_end = (int)((long long)total_it * (split + 1) / p.splits);
  const int nit = it_end - it_begin;

  double acc[MT][NT][2];
#pragma unroll
  for (int i = 0; i < MT; i++)
#pragma unroll
    for (int j = 0; j < NT; j++) acc[i][j][0] = acc[i][j][1] = 0.0;

  auto issue = [&](int li) {   // li = local iteration index
    if (li < nit) {
      int it = it_begin + li;
      int kb = it / ktiles, kt = it - kb * ktiles;
      int st = li % STAGES;
      load_tile<BM, BK, NTHREADS, AKM, AL16>(sA + st * A_STAGE, Ab + (long long)kb * p.sAk, p.lda, m0, p.M, kt * BK, p.K, tid);
      load_tile<BN, BK, NTHREADS, BKM, AL16>(sB + st * B_STAGE, Bb + (long long)kb * p.sBk, p.ldb, n0, p.N, kt * BK, p.K, tid);
    }
    cp_async_commit();
  };

#pragma unroll
  for (int s = 0; s < STAGES - 1; s++) issue(s);

  for (int li = 0; li < nit; li++) {
    cp_async_wait<STAGES - 2>();
    __syncthreads();
    issue(li + STAGES - 1);
    const double* a_s = sA + (li % STAGES) * A_STAGE;
    const double* b_s = sB + (li % STAGES) * B_STAGE;
#pragma unroll
    for (int kb8 = 0; kb8 < BK / 8; kb8++) {
      double af[MT][2], bf[NT][2];
#pragma unroll
      for (int i = 0; i < MT; i++) {
        int r = wm * WTM + i * 8 + g;
        if (AKM) {
          double2 v = *reinterpret_cast<const double2*>(a_s + (kb8 * BM + r) * 8 + 2 * t);
          af[i][0] = v.x; af[i][1] = v.y;
        } else {
          af[i][0] = a_s[(kb8 * 8 + 2 * t) * (BM + 2) + r];
          af[i][1] = a_s[(kb8 * 8 + 2 * t + 1) * (BM + 2) + r];
        }
      }
#pragma unroll
      for (int j = 0; j < NT; j++) {
        int r = wn * WTN + j * 8 + g;
        if (BKM) {
          double2 v = *reinterpret_cast<const double2*>(b_s + (kb8 * BN + r) * 8 + 2 * t);
          bf[j][0] = v.x; bf[j][1] = v.y;
        } else {
          bf[j][0] = b_s[(kb8 * 8 + 2 * t) * (BN + 2) + r];
          bf[j][1] = b_s[(kb8 * 8 + 2 * t + 1) * (BN + 2) + r];
        }
      }
#pragma unroll
      for (int h = 0; h < 2; h++)
#pragma unroll
        for (int i = 0; i < MT; i++)
#pragma unroll
          for (int j = 0; j < NT; j++) dmma884(acc[i][j][0], acc[i][j][1], af[i][h], bf[j][h]);
    }
  }
  cp_async_wait<0>();

  // epilogue
  const bool partial = p.splits > 1;
  double* Cb = p.C + (long long)b * p.sCb + (partial ? (long long)split * p.sCs : 0);
  const double* auxb = p.aux ? p.aux + (long long)b * p.sAuxb : nullptr;
  const bool vec = ((p.ldc & 1) == 0) && ((reinterpret_cast<uintptr_t>(Cb) & 15) == 0);
#pragma unroll
  for (int i = 0; i < MT; i++) {
    int m = m0 + wm * WTM + i * 8 + g;
    if (m >= p.M) continue;
#pragma unroll
    for (int j = 0; j < NT; j++) {
      int n = n0 + wn * WTN + j * 8 + 2 * t;
      if (n >= p.N) continue;
      double v0 = acc[i][j][0], v1 = acc[i][j][1];
      bool two = (n + 1 < p.N);
      if (!partial) {
        v0 *= p.alpha; v1 *= p.alpha;
        if (auxb) {
          v0 *= auxb[(long long)m * p.ldaux + n];
          if (two) v1 *= auxb[(long long)m * p.ldaux + n + 1];
        }
      }
      double* c = Cb + (long long)m * p.ldc + n;
      if (!partial && p.beta != 0.0) {
        v0 += p.beta * c[0];
        if (two) v1 += p.beta * c[1];
      }
      if (two && vec) {
        *reinterpret_cast<double2*>(c) = make_double2(v0, v1);
      } else {
        c[0] = v0;
        if (two) c[1] = v1;
      }
    }
  }
}

// dst = alpha * (sum_s part_s) (.* aux) + beta * dst, summed in split order (deterministic).
// part is laid out [split][batch][M][N] densely.
struct ReduceParams {
  const double* part; double* dst; const double* aux;
  int M, N, batch, splits;
  long long ldd, sDb, ldaux, sAuxb;
  double alpha, beta;
};
__global__ void reduce_splits_kernel(const ReduceParams p) {
  const long long per = (long long)p.batch * p.M * p.N;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < per; idx += (long long)gridDim.x * blockDim.x) {
    int n = (int)(idx % p.N);
    long long r = idx / p.N;
    int m = (int)(r % p.M);
    int b = (int)(r / p.M);
    double s = 0.0;
    for (int sp = 0; sp < p.splits; sp++) s += p.part[(long long)sp * per + idx];
    s *= p.alpha;
    if (p.aux) s *= p.aux[(long long)b * p.sAuxb + (long long)m * p.ldaux + n];
    double* d = p.dst + (long long)b * p.sDb + (long long)m * p.ldd + n;
    if (p.beta != 0.0) s += p.beta * *d;
    *d = s;
  }
}

}  // namespace thc
