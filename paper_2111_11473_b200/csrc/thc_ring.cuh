// Alg.7 lines 12-19 fused into one kernel for o <= 64:
//
//     FYT^P[j][I] = sum_J ( E^P[I][J] * V[I][J] ) Yo[j][J] ,      E^P[I][J] = sum_i YoT[I][i] RYT^P[J][i]
//
// (E = Yo^T R^P Yv, F = E .* V, and the first half of G^P = Yo F^T Yv^T).  E is NX x NX per grid point P and only ever
// feeds the Hadamard product and the next contraction, so it is never written to HBM: per 128-row I-tile the kernel
// walks over 32-column J-tiles, forms the E tile with DMMA (K = o), multiplies it by the V tile in registers and uses
// the product fragments directly as the A operand of the second DMMA chain (K = J).  No data movement is needed
// between the two chains: a C fragment holds columns 2t, 2t+1 of an 8-wide block, and the second chain simply takes its
// two k4 steps as k = 2t + h, the same k order the shared-memory operand layout [k/8][row][8] already uses.
// Same structure as a fused attention kernel with the softmax replaced by the fixed weights V_IJ.
//
// CTA = 256 threads = 8 warps, warp w owns rows 16w .. 16w+15 of the I-tile (2 m-tiles).  Registers: Q fragments of the
// warp's rows (loaded once), 16 FP64 E accumulators, 4*KT output accumulators (KT = ceil(o/8)).  Shared memory: 3-stage
// cp.async ring of {V tile 128 x 32 (pitch 40: rows g, g+1 fall into different bank halves), K tile [KT][32][8],
// Yo tile [4][8 KT][8]}.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "thc_gemm.cuh"

namespace thc {

constexpr int RG_BM = 128, RG_BN = 32, RG_STAGES = 3, RG_VPITCH = 40, RG_THREADS = 256;
__host__ __device__ constexpr int ring_stage_doubles(int KT) { return RG_BM * RG_VPITCH + KT * RG_BN * 8 + (RG_BN / 8) * (8 * KT) * 8; }
__host__ __device__ constexpr int ring_smem_bytes(int KT) { return RG_STAGES * ring_stage_doubles(KT) * 8; }

struct RingParams {
  const double* YoT;   // [NX][o]
  const double* RYT;   // [npb][NX][o]
  const double* V;     // [NX][NX]
  const double* Yo;    // [o][NX]
  double* FYT;         // [npb][o][NX]
  int NX, o, npb;
};

template <int KT, bool AL16>
__global__ void __launch_bounds__(RG_THREADS, 1) ring_fused_kernel(const RingParams p) {
  constexpr int O8 = 8 * KT, NT = RG_BN / 8;
  constexpr int STAGE = ring_stage_doubles(KT);
  constexpr int OFF_K = RG_BM * RG_VPITCH, OFF_Y = OFF_K + KT * RG_BN * 8;
  extern __shared__ __align__(16) double smem[];

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, g = lane >> 2, t = lane & 3;
  const int I0 = blockIdx.x * RG_BM;
  const int NX = p.NX, o = p.o;
  const double* RYT = p.RYT + (long long)blockIdx.y * NX * o;
  double* FYT = p.FYT + (long long)blockIdx.y * NX * o;
  const int nJ = (NX + RG_BN - 1) / RG_BN;

  // ---- fetch of one J-tile into a stage (zero-filled outside the arrays) ----------------------------------------------
  auto copy2 = [&](double* dst, const double* src, int n_ok) {      // two doubles, n_ok of them valid
    if (AL16) {
      cp_async16(dst, src, n_ok * 8);
    } else {
      cp_async8(dst, src, n_ok >= 1 ? 8 : 0);
      cp_async8(dst + 1, n_ok >= 2 ? src + 1 : src, n_ok >= 2 ? 8 : 0);
    }
  };
  auto fetch = [&](int jt) {
    if (jt < nJ) {
      double* st = smem + (jt % RG_STAGES) * STAGE;
      const int J0 = jt * RG_BN;
      // V tile: rows I0 .. I0+127, cols J0 .. J0+31
      for (int c = tid; c < RG_BM * RG_BN / 2; c += RG_THREADS) {
        const int r = c / (RG_BN / 2), cc = (c % (RG_BN / 2)) * 2;
        const int row = I0 + r, col = J0 + cc;
        const int n_ok = row < NX ? max(0, min(2, NX - col)) : 0;
        copy2(st + r * RG_VPITCH + cc, p.V + (n_ok ? (long long)row * NX + col : 0), n_ok);
      }
      // K tile: B(n = J, k = i) = RYT[J][i]  ->  [kb][n][8]
      for (int c = tid; c < KT * RG_BN * 4; c += RG_THREADS) {
        const int kb = c / (RG_BN * 4), rem = c % (RG_BN * 4), n = rem / 4, cc = (rem % 4) * 2;
        const int J = J0 + n, k = kb * 8 + cc;
        const int n_ok = J < NX ? max(0, min(2, o - k)) : 0;
        copy2(st + OFF_K + (kb * RG_BN + n) * 8 + cc, RYT + (n_ok ? (long long)J * o + k : 0), n_ok);
      }
      // Yo tile: B(n = j, k = J) = Yo[j][J]  ->  [kb][n][8], kb over the 4 k8-blocks of the J-tile
      for (int c = tid; c < NT * O8 * 4; c += RG_THREADS) {
        const int kb = c / (O8 * 4), rem = c % (O8 * 4), n = rem / 4, cc = (rem % 4) * 2;
        const int J = J0 + kb * 8 + cc;
        const int n_ok = n < o ? max(0, min(2, NX - J)) : 0;
        copy2(st + OFF_Y + (kb * O8 + n) * 8 + cc, p.Yo + (n_ok ? (long long)n * NX + J : 0), n_ok);
      }
    }
    cp_async_commit();
  };
#pragma unroll
  for (int s = 0; s < RG_STAGES - 1; s++) fetch(s);

  // ---- Q fragments of this warp's 16 rows: A(m = I, k = i) = YoT[I][i], k = 8 kb + 2t + h ------------------------------
  double qf[2][KT][2];
#pragma unroll
  for (int i = 0; i < 2; i++) {
    const int row = I0 + warp * 16 + i * 8 + g;
#pragma unroll
    for (int kb = 0; kb < KT; kb++)
#pragma unroll
      for (int h = 0; h < 2; h++) {
        const int k = kb * 8 + 2 * t + h;
        qf[i][kb][h] = (row < NX && k < o) ? p.YoT[(long long)row * o + k] : 0.0;
      }
  }
  double oacc[2][KT][2];
#pragma unroll
  for (int i = 0; i < 2; i++)
#pragma unroll
    for (int jj = 0; jj < KT; jj++) oacc[i][jj][0] = oacc[i][jj][1] = 0.0;

  const bool fetch_first = ((warp >> 2) & 1) == 0;       // stagger the address work of the two warps of an SM sub-partition
  for (int jt = 0; jt < nJ; jt++) {
    cp_async_wait<RG_STAGES - 2>();
    __syncthreads();
    if (fetch_first) fetch(jt + RG_STAGES - 1);
    const double* st = smem + (jt % RG_STAGES) * STAGE;
    // chain 1: E tile (16 rows x 32 cols per warp), K = o
    double sacc[2][NT][2];
#pragma unroll
    for (int i = 0; i < 2; i++)
#pragma unroll
      for (int j = 0; j < NT; j++) sacc[i][j][0] = sacc[i][j][1] = 0.0;
#pragma unroll
    for (int kb = 0; kb < KT; kb++) {
#pragma unroll
      for (int j = 0; j < NT; j++) {
        const double2 b = *reinterpret_cast<const double2*>(st + OFF_K + (kb * RG_BN + j * 8 + g) * 8 + 2 * t);
#pragma unroll
        for (int i = 0; i < 2; i++) {
          dmma884(sacc[i][j][0], sacc[i][j][1], qf[i][kb][0], b.x);
          dmma884(sacc[i][j][0], sacc[i][j][1], qf[i][kb][1], b.y);
        }
      }
    }
    if (!fetch_first) fetch(jt + RG_STAGES - 1);
    // F = E .* V
#pragma unroll
    for (int i = 0; i < 2; i++)
#pragma unroll
      for (int j = 0; j < NT; j++) {
        const double2 vv = *reinterpret_cast<const double2*>(st + (warp * 16 + i * 8 + g) * RG_VPITCH + j * 8 + 2 * t);
        sacc[i][j][0] *= vv.x; sacc[i][j][1] *= vv.y;
      }
    // chain 2: O += F . Yo^T, K = the 32 columns J of this tile; k8-block j of the chain is n-tile j of chain 1
#pragma unroll
    for (int j = 0; j < NT; j++) {
#pragma unroll
      for (int jj = 0; jj < KT; jj++) {
        const double2 b = *reinterpret_cast<const double2*>(st + OFF_Y + (j * O8 + jj * 8 + g) * 8 + 2 * t);
#pragma unroll
        for (int i = 0; i < 2; i++) {
          dmma884(oacc[i][jj][0], oacc[i][jj][1], sacc[i][j][0], b.x);
          dmma884(oacc[i][jj][0], oacc[i][jj][1], sacc[i][j][1], b.y);
        }
      }
    }
  }
  cp_async_wait<0>();

  // ---- FYT[j][I] ---------------------------------------------------------------------------------------------------------
#pragma unroll
  for (int i = 0; i < 2; i++) {
    const int row = I0 + warp * 16 + i * 8 + g;
    if (row >= NX) continue;
#pragma unroll
    for (int jj = 0; jj < KT; jj++) {
      const int col = jj * 8 + 2 * t;
      if (col < o) FYT[(long long)col * NX + row] = oacc[i][jj][0];
      if (col + 1 < o) FYT[(long long)(col + 1) * NX + row] = oacc[i][jj][1];
    }
  }
}

}  // namespace thc
