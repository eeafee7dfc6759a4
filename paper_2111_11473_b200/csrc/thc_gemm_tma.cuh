// FP64 DMMA GEMM, TMA-fed and persistent: the kernel behind the large K-major x K-major products of the GEMM chains
// (half-transforms of the Cholesky vectors, D^L = C^L Z, sigma1 += D^L C^L^T, the E_I / F_I / G_I feeders of Alg.6, the
// chains of Alg.7; "rate limiting step ... cuBLAS", here hand-written).  Same contract as dgemm_kernel
// (thc_gemm.cuh: batch, strided second K loop, split-K partials, alpha / beta / aux / transposed copy, upper-only tiles).
//
// B200 design
//   * operands arrive by TMA (cp.async.bulk.tensor.4d: coordinates k, row, k-batch, batch) as boxes of 8 k x ROWS rows,
//     i.e. exactly the [k/8][row][8] shared-memory layout whose 16-byte fragment loads are bank-conflict free; K tails
//     and ragged row tiles are zero-filled by the TMA unit, so the k loop has no bounds arithmetic at all;
//   * one producer warp (one elected lane) issues the boxes and runs ahead through a STAGES-deep ring of full / empty
//     mbarriers; the consumer warps never touch addresses of the operands: their issue slots go to DMMA.8x8x4 and LDS.128.
//     The producer sits in a warpgroup of its own that gives its registers back (setmaxnreg.dec 40) so that the two
//     consumer warpgroups can hold a 128 x 128 FP64 accumulator tile plus double-buffered fragments (setmaxnreg.inc 232);
//   * persistent CTAs (one per SM) walk a static tile list; the ring runs across tile boundaries, so the loads of the
//     next tile are in flight during the epilogue of the current one, and because there is no CTA-wide barrier in the
//     main loop the warps drift apart by up to STAGES k-tiles: while one warp of an SM sub-partition stores its
//     fragments the other one keeps the FP64 tensor pipe busy (matters for the small-K products, K = o).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include "thc_gemm.cuh"
#include "thc_triple.cuh"      // mbarrier / TMA helpers

namespace thc {

constexpr int TG_BK = 16;

__device__ __forceinline__ void tma_load_4d(uint32_t dst, const CUtensorMap* map, int c0, int c1, int c2, int c3, uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
      ::"r"(dst), "l"(reinterpret_cast<uint64_t>(map)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(bar) : "memory");
}

__host__ __device__ constexpr int tg_smem_bytes(int BM, int BN, int STAGES) {
  return STAGES * (BM + BN) * TG_BK * 8 + 2 * STAGES * 8 + 128 /* alignment slack */;
}

// Tile t of the launch -> (batch, split, tile_m, tile_n).  Order: tile_n fastest, then tile_m, then split, then batch, so
// that the CTAs running at the same time share operand rows in L2.  upper_only (square tile grid): only tiles with
// tile_n >= tile_m exist, enumerated row by row.
struct TgTile { int b, split, tm, tn; };
__device__ __forceinline__ TgTile tg_decode(long long t, int tiles_m, int tiles_n, int splits, int upper) {
  TgTile r;
  const long long per = upper ? (long long)tiles_m * (tiles_m + 1) / 2 : (long long)tiles_m * tiles_n;
  const long long bs = t / per;
  long long rem = t - bs * per;
  r.split = (int)(bs % splits);
  r.b = (int)(bs / splits);
  if (!upper) {
    r.tm = (int)(rem / tiles_n);
    r.tn = (int)(rem - (long long)r.tm * tiles_n);
  } else {
    // row tm holds tiles_m - tm tiles; rows before it hold tm * tiles_m - tm (tm - 1) / 2
    int tm = (int)(((2.0 * tiles_m + 1.0) - sqrt((2.0 * tiles_m + 1.0) * (2.0 * tiles_m + 1.0) - 8.0 * (double)rem)) * 0.5);
    while (tm > 0 && (long long)tm * tiles_m - (long long)tm * (tm - 1) / 2 > rem) tm--;
    while ((long long)(tm + 1) * tiles_m - (long long)(tm + 1) * tm / 2 <= rem) tm++;
    r.tm = tm;
    r.tn = tm + (int)(rem - ((long long)tm * tiles_m - (long long)tm * (tm - 1) / 2));
  }
  return r;
}

constexpr int TG_THREADS = 384;      // 8 consumer warps (two warpgroups) + the producer's warpgroup

template <int BM, int BN, int WM, int WN, int STAGES>
__global__ void __launch_bounds__(TG_THREADS, 1)
dgemm_tma_kernel(const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapB, const GemmParams p) {
  constexpr int NCW = WM * WN;                                   // consumer warps
  static_assert(NCW == 8, "two consumer warpgroups");
  constexpr int WTM = BM / WM, WTN = BN / WN, MT = WTM / 8, NT = WTN / 8;
  constexpr int A_STAGE = BM * TG_BK, B_STAGE = BN * TG_BK;      // doubles
  constexpr int STAGE_BYTES = (A_STAGE + B_STAGE) * 8;
  extern __shared__ uint8_t tg_smem_raw[];
  const uint32_t base = (smem_u32(tg_smem_raw) + 127u) & ~127u;
  const double* ring = reinterpret_cast<const double*>(tg_smem_raw + (base - smem_u32(tg_smem_raw)));
  const uint32_t bar_full = base + STAGES * STAGE_BYTES, bar_empty = bar_full + STAGES * 8;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int tiles_m = (p.M + BM - 1) / BM, tiles_n = (p.N + BN - 1) / BN;
  const int ktiles = (p.K + TG_BK - 1) / TG_BK;
  const int total_it = p.kbatch * ktiles;
  const long long per = p.upper_only ? (long long)tiles_m * (tiles_m + 1) / 2 : (long long)tiles_m * tiles_n;
  const long long n_tiles = per * p.splits * p.batch;

  if (tid == 0) {
    for (int s = 0; s < STAGES; s++) { mbar_init(bar_full + 8 * s, 1); mbar_init(bar_empty + 8 * s, NCW); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  if (warp >= NCW) {
    // ---- producer: one lane walks the same tile list as the consumers and keeps the ring full -------------------------
    asm volatile("setmaxnreg.dec.sync.aligned.u32 40;");
    if (warp != NCW || lane != 0) return;
    long long fill = 0;
    for (long long t = blockIdx.x; t < n_tiles; t += gridDim.x) {
      const TgTile tl = tg_decode(t, tiles_m, tiles_n, p.splits, p.upper_only);
      const int it_begin = (int)((long long)total_it * tl.split / p.splits);
      const int it_end = (int)((long long)total_it * (tl.split + 1) / p.splits);
      int kb = it_begin / ktiles, kt = it_begin - kb * ktiles;
      const int bA = p.sAb ? tl.b : 0, bB = p.sBb ? tl.b : 0;       // a broadcast operand has extent 1 in that dimension
      for (int it = it_begin; it < it_end; it++, fill++) {
        const int s = (int)(fill % STAGES);
        if (fill >= STAGES) mbar_wait(bar_empty + 8 * s, (uint32_t)(((fill / STAGES) - 1) & 1));
        const uint32_t dst = base + s * STAGE_BYTES, bf = bar_full + 8 * s;
        mbar_expect_tx(bf, STAGE_BYTES);
        const int k0 = kt * TG_BK, kbA = p.sAk ? kb : 0, kbB = p.sBk ? kb : 0;
        tma_load_4d(dst, &mapA, k0, tl.tm * BM, kbA, bA, bf);
        tma_load_4d(dst + BM * 64, &mapA, k0 + 8, tl.tm * BM, kbA, bA, bf);
        tma_load_4d(dst + A_STAGE * 8, &mapB, k0, tl.tn * BN, kbB, bB, bf);
        tma_load_4d(dst + A_STAGE * 8 + BN * 64, &mapB, k0 + 8, tl.tn * BN, kbB, bB, bf);
        if (++kt == ktiles) { kt = 0; kb++; }
      }
    }
    return;
  }

  // ---- consumers ---------------------------------------------------------------------------------------------------------
  asm volatile("setmaxnreg.inc.sync.aligned.u32 232;");
  const int g = lane >> 2, t4 = lane & 3;
  const int wm = warp / WN, wn = warp % WN;
  int st = 0;
  uint32_t par = 0;
  for (long long t = blockIdx.x; t < n_tiles; t += gridDim.x) {
    const TgTile tl = tg_decode(t, tiles_m, tiles_n, p.splits, p.upper_only);
    const int nit = (int)((long long)total_it * (tl.split + 1) / p.splits) - (int)((long long)total_it * tl.split / p.splits);
    double acc[MT][NT][2];
#pragma unroll
    for (int i = 0; i < MT; i++)
#pragma unroll
      for (int j = 0; j < NT; j++) acc[i][j][0] = acc[i][j][1] = 0.0;

    for (int li = 0; li < nit; li++) {
      mbar_wait(bar_full + 8 * st, par);
      const double* a_s = ring + st * (A_STAGE + B_STAGE);
      const double* b_s = a_s + A_STAGE;
      double af[2][MT][2], bf[2][NT][2];
      auto load_frags = [&](int buf, int kb8) {
#pragma unroll
        for (int i = 0; i < MT; i++) {
          const double2 v = *reinterpret_cast<const double2*>(a_s + (kb8 * BM + wm * WTM + i * 8 + g) * 8 + 2 * t4);
          af[buf][i][0] = v.x; af[buf][i][1] = v.y;
        }
#pragma unroll
        for (int j = 0; j < NT; j++) {
          const double2 v = *reinterpret_cast<const double2*>(b_s + (kb8 * BN + wn * WTN + j * 8 + g) * 8 + 2 * t4);
          bf[buf][j][0] = v.x; bf[buf][j][1] = v.y;
        }
      };
      load_frags(0, 0);
#pragma unroll
      for (int kb8 = 0; kb8 < TG_BK / 8; kb8++) {
        if (kb8 + 1 < TG_BK / 8) load_frags((kb8 + 1) & 1, kb8 + 1);
#pragma unroll
        for (int h = 0; h < 2; h++)
#pragma unroll
          for (int i = 0; i < MT; i++)
#pragma unroll
            for (int j = 0; j < NT; j++) dmma884(acc[i][j][0], acc[i][j][1], af[kb8 & 1][i][h], bf[kb8 & 1][j][h]);
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(bar_empty + 8 * st);
      if (++st == STAGES) { st = 0; par ^= 1; }
    }

    // ---- epilogue (same semantics as dgemm_kernel) -----------------------------------------------------------------------
    const int m0 = tl.tm * BM, n0 = tl.tn * BN, b = tl.b;
    const bool partial = p.splits > 1;
    double* Cb = p.C + (long long)b * p.sCb + (partial ? (long long)tl.split * p.sCs : 0);
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
        const int n = n0 + wn * WTN + j * 8 + 2 * t4;
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
        const int n = n0 + wn * WTN + j * 8 + 2 * t4;
        if (n >= p.N) continue;
        const bool two = (n + 1 < p.N);
        const double r0 = acc[i][j][0] * alpha, r1 = acc[i][j][1] * alpha;
        if (p.Ct != nullptr && !partial) {
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
}

}  // namespace thc
