// FP64 DMMA GEMM for sm_100a: the one kernel every GEMM chain of the THC-RR-CCSD residual runs on.
//
//   C_b[m][n] = alpha * ( sum_{kb < kbatch} sum_{k < K} A_{b,kb}(m,k) * B_{b,kb}(n,k) ) (.* aux_b[m][n]) + beta * C_b[m][n]
//
// A(m,k) = A[m*lda + k] ("K-major") or A[k*lda + m] ("M-major"); likewise B(n,k).  `kbatch` is a second,
// strided K loop (sum over Cholesky vectors of D^L C^L^T, Alg.1 line 15 l.524); `Ct` is an optional transposed copy
// of the product (Alg.6 needs G_I in both orientations); `splits` cuts the
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
  double* Ct; long long ldct, sCtb;   // optional second output: Ct_b[n][m] = alpha * (A B^T)[m][n] (no aux, no beta)
  int upper_only;                     // symmetric product: CTAs whose tile lies strictly below the diagonal do nothing
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

// Per-thread state for copying one BK-deep slab of an operand tile (ROWS rows of an operand with `nrows` rows) into shared
// memory.  Every index computation (chunk -> row / k offset, row bounds, smem offset) is done once in init(); issuing a
// slab costs a pointer add and a K-tail clamp per 16-byte chunk, so the warps spend their issue slots on DMMA.
//   K-major operand: smem [BK/8][ROWS][8], global element (r, k) at g[r*ld + k]
//   M/N-major      : smem [BK][ROWS+2],    global element (r, k) at g[k*ld + r]
template <int ROWS, int BK, int NTHREADS, bool KMAJOR, bool AL16>
struct TileLoader {
  static constexpr int CHUNKS = ROWS * BK / 2;
  static constexpr int NCH = (CHUNKS + NTHREADS - 1) / NTHREADS;
  long long goff[NCH];   // global offset of the chunk in k-tile 0 (doubles)
  int soff[NCH];         // shared offset inside a stage (doubles)
  int kofs[NCH];         // k offset inside the tile
  int bytes[NCH];        // bytes the chunk may copy as far as the row bound is concerned (0, 8 or 16)
  long long kstep;       // global offset between consecutive k-tiles
  __device__ __forceinline__ void init(long long ld, int row0, int nrows, int tid) {
#pragma unroll
    for (int q = 0; q < NCH; q++) {
      const int c = tid + q * NTHREADS;
      if (KMAJOR) {
        const int kb8 = c / (ROWS * 4), rem = c % (ROWS * 4), r = rem / 4, cc = rem % 4;
        const int row = row0 + r;
        const bool ok = c < CHUNKS && row < nrows;
        soff[q] = (kb8 * ROWS + r) * 8 + cc * 2;
        kofs[q] = kb8 * 8 + cc * 2;
        goff[q] = (ok ? (long long)row * ld : 0) + kofs[q];
        bytes[q] = ok ? 16 : 0;
      } else {
        const int kk = c / (ROWS / 2), cc = c % (ROWS / 2);
        const int row = row0 + cc * 2;
        const bool ok = c < CHUNKS;
        soff[q] = kk * (ROWS + 2) + cc * 2;
        kofs[q] = kk;
        goff[q] = (long long)kk * ld + (row < nrows ? row : 0);
        bytes[q] = ok ? max(0, min(2, nrows - row)) * 8 : 0;
      }
    }
    kstep = KMAJOR ? BK : (long long)BK * ld;
  }
  // copy the slab of k-tile kt of operand base `g` into stage `s`
  __device__ __forceinline__ void issue(double* s, const double* __restrict__ g, int kt, int K) const {
    const int k0 = kt * BK;
    const double* gk = g + (long long)kt * kstep;
    if (k0 + BK <= K) {                                      // full k-tile (all but the last): no K-tail arithmetic
#pragma unroll
      for (int q = 0; q < NCH; q++) {
        if (NCH * NTHREADS != CHUNKS && threadIdx.x + q * NTHREADS >= CHUNKS) continue;
        const double* src = gk + goff[q];                    // rows beyond the operand point at row 0 and copy 0 bytes
        double* dst = s + soff[q];
        if (AL16) {
          cp_async16(dst, src, bytes[q]);
        } else {
          cp_async8(dst, src, bytes[q] >= 8 ? 8 : 0);
          cp_async8(dst + 1, bytes[q] >= 16 ? src + 1 : src, bytes[q] >= 16 ? 8 : 0);
        }
      }
      return;
    }
#pragma unroll
    for (int q = 0; q < NCH; q++) {
      if (NCH * NTHREADS != CHUNKS && bytes[q] == 0 && threadIdx.x + q * NTHREADS >= CHUNKS) continue;
      const int krem = K - (k0 + kofs[q]);                   // k values left from this chunk's first k
      int nb;
      if (KMAJOR) nb = krem >= 2 ? bytes[q] : (krem == 1 ? min(bytes[q], 8) : 0);
      else nb = krem >= 1 ? bytes[q] : 0;
      const double* src = nb > 0 ? gk + goff[q] : g;
      double* dst = s + soff[q];
      if (AL16) {
        cp_async16(dst, src, nb);
      } else {
        cp_async8(dst, src, nb >= 8 ? 8 : 0);
        cp_async8(dst + 1, nb >= 16 ? src + 1 : src, nb >= 16 ? 8 : 0);
      }
    }
  }
};

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
  if (p.upper_only && n0 + BN <= m0) return;       // whole tile has n < m: the caller mirrors it from the upper triangle
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

  TileLoader<BM, BK, NTHREADS, AKM, AL16> ldA;
  TileLoader<BN, BK, NTHREADS, BKM, AL16> ldB;
  ldA.init(p.lda, m0, p.M, tid);
  ldB.init(p.ldb, n0, p.N, tid);
  // (kb, kt) of the next slab to fetch, advanced incrementally (no division in the loop)
  int f_kb = it_begin / ktiles, f_kt = it_begin - f_kb * ktiles, f_li = 0;
  auto issue = [&]() {
    if (f_li < nit) {
      const int st = f_li % STAGES;
      ldA.issue(sA + st * A_STAGE, Ab + (long long)f_kb * p.sAk, f_kt, p.K);
      ldB.issue(sB + st * B_STAGE, Bb + (long long)f_kb * p.sBk, f_kt, p.K);
      if (++f_kt == ktiles) { f_kt = 0; f_kb++; }
    }
    f_li++;
    cp_async_commit();
  };

#pragma unroll
  for (int s = 0; s < STAGES - 1; s++) issue();

  for (int li = 0; li < nit; li++) {
    cp_async_wait<STAGES - 2>();
    __syncthreads();
    // the two warps that share an SM sub-partition (w and w + 4) fetch at different times, so that one of them is always
    // issuing DMMAs while the other does its cp.async address work
    const bool fetch_first = ((warp >> 2) & 1) == 0;
    if (fetch_first) issue();
    const double* a_s = sA + (li % STAGES) * A_STAGE;
    const double* b_s = sB + (li % STAGES) * B_STAGE;
    // fragments of k-block kb8 (8 k = two k4 steps h: k = 2t + h), double-buffered in registers so that the loads of
    // block kb8 + 1 are in flight while the 2 * MT * NT DMMAs of block kb8 issue
    double af[2][MT][2], bf[2][NT][2];
    auto load_frags = [&](int buf, int kb8) {
#pragma unroll
      for (int i = 0; i < MT; i++) {
        int r = wm * WTM + i * 8 + g;
        if (AKM) {
          double2 v = *reinterpret_cast<const double2*>(a_s + (kb8 * BM + r) * 8 + 2 * t);
          af[buf][i][0] = v.x; af[buf][i][1] = v.y;
        } else {
          af[buf][i][0] = a_s[(kb8 * 8 + 2 * t) * (BM + 2) + r];
          af[buf][i][1] = a_s[(kb8 * 8 + 2 * t + 1) * (BM + 2) + r];
        }
      }
#pragma unroll
      for (int j = 0; j < NT; j++) {
        int r = wn * WTN + j * 8 + g;
        if (BKM) {
          double2 v = *reinterpret_cast<const double2*>(b_s + (kb8 * BN + r) * 8 + 2 * t);
          bf[buf][j][0] = v.x; bf[buf][j][1] = v.y;
        } else {
          bf[buf][j][0] = b_s[(kb8 * 8 + 2 * t) * (BN + 2) + r];
          bf[buf][j][1] = b_s[(kb8 * 8 + 2 * t + 1) * (BN + 2) + r];
        }
      }
    };
    load_frags(0, 0);
#pragma unroll
    for (int kb8 = 0; kb8 < BK / 8; kb8++) {
      if (kb8 + 1 < BK / 8) load_frags((kb8 + 1) & 1, kb8 + 1);
#pragma unroll
      for (int h = 0; h < 2; h++)
#pragma unroll
        for (int i = 0; i < MT; i++)
#pragma unroll
          for (int j = 0; j < NT; j++) dmma884(acc[i][j][0], acc[i][j][1], af[kb8 & 1][i][h], bf[kb8 & 1][j][h]);
      if (kb8 == 0 && !fetch_first) issue();
    }
  }
  cp_async_wait<0>();

  // epilogue.  The operands of a row of fragments (aux values, old C values for beta != 0) are loaded for all NT
  // fragments first and only then combined and stored, so that their latencies overlap (one dependent load per stored
  // fragment made the small-K products with an aux operand epilogue-bound).
  const bool partial = p.splits > 1;
  double* Cb = p.C + (long long)b * p.sCb + (partial ? (long long)split * p.sCs : 0);
  const double* auxb = (p.aux && !partial) ? p.aux + (long long)b * p.sAuxb : nullptr;
  const bool use_beta = !partial && p.beta != 0.0;
  const bool vec = ((p.ldc & 1) == 0) && ((reinterpret_cast<uintptr_t>(Cb) & 15) == 0);
  const bool vec_aux = auxb && ((p.ldaux & 1) == 0) && ((reinterpret_cast<uintptr_t>(auxb) & 15) == 0);
  const double alpha = partial ? 1.0 : p.alpha;
#pragma unroll
  for (int i = 0; i < MT; i++) {
    const int m = m0 + wm * WTM + i * 8 + g;
    if (m >= p.M) continue;
    double ax[NT][2], cx[NT][2];
#pragma unroll
    for (int j = 0; j < NT; j++) {
      const int n = n0 + wn * WTN + j * 8 + 2 * t;
      ax[j][0] = ax[j][1] = 1.0;
      cx[j][0] = cx[j][1] = 0.0;
      if (n >= p.N) continue;
      const bool two = (n + 1 < p.N);
      if (auxb) {
        const double* a = auxb + (long long)m * p.ldaux + n;
        if (two && vec_aux) { const double2 v = *reinterpret_cast<const double2*>(a); ax[j][0] = v.x; ax[j][1] = v.y; }
        else { ax[j][0] = a[0]; if (two) ax[j][1] = a[1]; }
      }
      if (use_beta) {
        const double* c = Cb + (long long)m * p.ldc + n;
        if (two && vec) { const double2 v = *reinterpret_cast<const double2*>(c); cx[j][0] = v.x; cx[j][1] = v.y; }
        else { cx[j][0] = c[0]; if (two) cx[j][1] = c[1]; }
      }
    }
#pragma unroll
    for (int j = 0; j < NT; j++) {
      const int n = n0 + wn * WTN + j * 8 + 2 * t;
      if (n >= p.N) continue;
      const bool two = (n + 1 < p.N);
      const double r0 = acc[i][j][0] * alpha, r1 = acc[i][j][1] * alpha;
      if (p.Ct != nullptr && !partial) {          // transposed copy: the bare product, before aux / beta
        double* ct = p.Ct + (long long)b * p.sCtb + (long long)n * p.ldct + m;
        ct[0] = r0;
        if (two) ct[p.ldct] = r1;
      }
      double v0 = r0 * ax[j][0], v1 = r1 * ax[j][1];
      if (use_beta) { v0 += p.beta * cx[j][0]; v1 += p.beta * cx[j][1]; }
      double* c = Cb + (long long)m * p.ldc + n;
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
  int skip_bm, skip_bn;     // upper-only product: elements of tiles (skip_bm x skip_bn) strictly below the diagonal are left alone
};
__global__ void reduce_splits_kernel(const ReduceParams p) {
  const long long per = (long long)p.batch * p.M * p.N;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < per; idx += (long long)gridDim.x * blockDim.x) {
    int n = (int)(idx % p.N);
    long long r = idx / p.N;
    int m = (int)(r % p.M);
    int b = (int)(r / p.M);
    if (p.skip_bm && (n / p.skip_bn + 1) * p.skip_bn <= (m / p.skip_bm) * p.skip_bm) continue;
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
