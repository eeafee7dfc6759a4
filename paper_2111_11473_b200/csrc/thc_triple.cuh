// Alg.6 line 11, the rate-limiting step of the THC ladder-type T2^2 terms ("implemented with a custom
// CUDA kernel", l.257):
//
//     H[p][q][r] (+)= sum_I ( E_I[p][q] F_I[p][r] + E_I[p][r] F_I[p][q] ) G_I[q][r]
//
// This is a three-way "triangle" product (every factor carries two of the three output indices and the summed index),
// not a dense contraction: it runs on the FP64 FMA pipe.  Work per (p,q,r,I):
//   the bracket s_I[p](q,r) is symmetric in (q,r), so a CTA that owns the block (p-tile, q-tile, r-tile) with the q-tile
//   outside the r-tile also owns the mirrored block (p-tile, r-tile, q-tile): s is formed once (DMUL + DFMA) and used
//   twice (2 DFMA) -> 2 FP64 instructions per (p,q,r,I) instead of 3.  CTAs whose q-tile lies inside their r-tile
//   ("diagonal") do the plain 3-instruction update of the direct block only.
//
// B200 design
//   * persistent CTAs (one per SM, 256 threads = 8 warps as 2p x 2q x 2r; lane = 2p x 4q x 4r; thread tile 4p x 2q x 4r
//     plus its mirror = 64 FP64 accumulators), CTA tile 16p x 16q x 32r (+ mirror 16p x 32r x 16q);
//   * operands are fetched by TMA (cp.async.bulk.tensor.3d, SWIZZLE_128B) as ten boxes of 16 x 16 x TP_IC FP64 values
//     (TP_IC = 2 grid points, 4 KB per box) into a TP_STAGES-deep shared-memory ring; full/empty mbarriers, no
//     __syncthreads in the I loop.  Thread 0 issues the boxes of stage j + TP_STAGES - 2 when it enters stage j (two
//     stages of slack on the empty barrier; its counters live in shared memory), so ~120 KB are in flight per SM.  The
//     mirrored block needs G_I[r][q]: it is read from the tile of G_I at (rows r-tile, columns q-tile) -- no transposed
//     copy of G exists (it would double the memory of the I-chunk, which at paper scale decides the block sizes);
//   * the 128-byte swizzle makes every 16-byte fragment load bank-conflict free.  The eight lanes of a quarter-warp are
//     four r offsets x two q offsets; the two q offsets are chosen 6 or 2 apart (q pairs 0/3 and 1/2 of the warp's four),
//     so that they differ both in bit 2 of the row (direct reads of G: rows q, chunks r) and in bit 0 of the 16-byte
//     chunk (transposed reads of G: rows r, chunks q) -- both read patterns hit eight different chunks;
//   * work items (p-tile, q-tile, r-tile) come from a host-built list ordered in groups of 8 p-tiles x 6 q-tiles x 3
//     r-tiles, so that the ~148 CTAs running at the same time share their operand tiles in L2.  That only works while
//     they run in step: long launches are cooperative and the CTAs wait for one another every ~16384 grid points of work
//     (TripleParams::gate); ungated they drift apart and two tiles out of three come from DRAM (2.9 TB/s, +100 W).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace thc {

constexpr int TP_PT = 16, TP_QT = 16, TP_RT = 32;
constexpr int TP_IC = 2;                                   // grid points per pipeline stage (one barrier round-trip per stage)
constexpr int TP_STAGES = 5, TP_LOOKAHEAD = TP_STAGES - 2;
constexpr int TP_SLICE_BYTES = 16 * 16 * 8;                // one 16x16 FP64 block of one grid point
constexpr int TP_BLK_BYTES = TP_IC * TP_SLICE_BYTES;       // one TMA box: 16 x 16 x TP_IC
constexpr int TP_STAGE_BYTES = 10 * TP_BLK_BYTES;          // EPQ FPQ EPR0 EPR1 FPR0 FPR1 GQR0 GQR1 GRQ0 GRQ1
constexpr int TP_SMEM_BYTES = TP_STAGES * TP_STAGE_BYTES + 1024 /* alignment slack */ + 2 * TP_STAGES * 8;
constexpr int TP_THREADS = 256;

struct TripleItem { int p0, q0, r0, diag; };

struct TripleParams {
  double* H;
  const TripleItem* items;
  int n_items;
  int nI, nPp, NPp;        // padded extents: nPp % 16 == 0, NPp % 32 == 0
  int accumulate;
  // Gate (0 = off): after every gate_every-th work item all CTAs of the (cooperative) launch wait for one another on the
  // counter *gate (zeroed before the launch).  CTAs that share operand tiles through the L2-ordered work list only hit in
  // L2 while they run in step; without a restoring force they drift apart by more than an L2 lifetime.
  unsigned int* gate;
  int gate_every;
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, int bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
      : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
  return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  while (!mbar_try_wait(bar, parity)) {}
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* map, int c0, int c1, int c2, uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
      ::"r"(dst), "l"(reinterpret_cast<uint64_t>(map)), "r"(c0), "r"(c1), "r"(c2), "r"(bar) : "memory");
}
__device__ __forceinline__ double2 lds128(const uint8_t* base, uint32_t off) {
  return *reinterpret_cast<const double2*>(base + off);
}


// One grid point of the register-tile update.  `sl` = the grid point's slice inside the stage (block b of the stage at
// sl + b * TP_BLK_BYTES).  hrq[a][b][c] accumulates H[p_a][r_c][q_b].
template <bool DIAG>
__device__ __forceinline__ void tp_update(const uint8_t* sl, const uint32_t (&offPQ)[4], const uint32_t (&offPR)[4],
                                          const uint32_t (&offQR)[2], uint32_t offT, double (&hqr)[4][2][4],
                                          double (&hrq)[4][2][4]) {
  double gqr[2][4], gt[2][4];            // gt[b][c] = G_I[r_c][q_b], from the tile of G_I at (rows r, columns q)
#pragma unroll
  for (int b = 0; b < 2; b++) {
    double2 g0 = lds128(sl, offQR[b]), g1 = lds128(sl, (offQR[b] ^ 64));
    gqr[b][0] = g0.x; gqr[b][1] = g0.y; gqr[b][2] = g1.x; gqr[b][3] = g1.y;
  }
  if (!DIAG) {
    // rows r_c = 2 lr + (c & 1) + 8 (c >> 1) of block 8 + wr; one 16-byte load gives (q_0, q_1) of a row.  offT is the
    // offset of row 2 lr; row 2 lr + 1 is at offT ^ 144 (next row, chunk bit 0 flipped by the swizzle), rows + 8 are
    // 1024 bytes further with the same swizzle phase.
    const double2 t0 = lds128(sl, offT), t1 = lds128(sl, offT ^ 144), t2 = lds128(sl, offT + 1024), t3 = lds128(sl, (offT ^ 144) + 1024);
    gt[0][0] = t0.x; gt[1][0] = t0.y; gt[0][1] = t1.x; gt[1][1] = t1.y;
    gt[0][2] = t2.x; gt[1][2] = t2.y; gt[0][3] = t3.x; gt[1][3] = t3.y;
  }
#pragma unroll
  for (int a = 0; a < 4; a++) {
    double2 e = lds128(sl, offPQ[a]), f = lds128(sl, TP_BLK_BYTES + offPQ[a]);
    double2 e0 = lds128(sl, offPR[a]), e1 = lds128(sl, (offPR[a] ^ 64));
    double2 f0 = lds128(sl, 2 * TP_BLK_BYTES + offPR[a]), f1 = lds128(sl, 2 * TP_BLK_BYTES + (offPR[a] ^ 64));
    const double epq[2] = {e.x, e.y}, fpq[2] = {f.x, f.y};
    const double epr[4] = {e0.x, e0.y, e1.x, e1.y}, fpr[4] = {f0.x, f0.y, f1.x, f1.y};
#pragma unroll
    for (int b = 0; b < 2; b++)
#pragma unroll
      for (int c = 0; c < 4; c++) {
        const double sv = fma(epr[c], fpq[b], epq[b] * fpr[c]);
        hqr[a][b][c] = fma(sv, gqr[b][c], hqr[a][b][c]);
        if (!DIAG) hrq[a][b][c] = fma(sv, gt[b][c], hrq[a][b][c]);
      }
  }
}

// E, F: tensor maps over [nI][nPp][NPp] (innermost NPp); G: over [nI][NPp][NPp]; box 16 x 16 x TP_IC, SWIZZLE_128B.
// Grid points beyond nI (odd nI) are zero-filled by the TMA unit and add nothing.
__global__ void __launch_bounds__(TP_THREADS, 1)
triple_product_kernel(const __grid_constant__ CUtensorMap mapE, const __grid_constant__ CUtensorMap mapF,
                      const __grid_constant__ CUtensorMap mapG, const TripleParams p) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t ring = (smem_u32(smem_raw) + 1023u) & ~1023u;          // 1024-byte aligned (swizzle atom)
  const uint8_t* ring_ptr = smem_raw + (ring - smem_u32(smem_raw));
  const uint32_t bar_full = ring + TP_STAGES * TP_STAGE_BYTES;
  const uint32_t bar_empty = bar_full + TP_STAGES * 8;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int wp = warp >> 2, wq = (warp >> 1) & 1, wr = warp & 1;
  // lane bits: 0-1 r offset, 2-3 q offset (pairs 0/3 and 1/2 inside a quarter-warp, see above), 4 p offset
  const int lp = lane >> 4, lq = ((lane >> 3) & 1) ^ (((lane >> 2) & 1) * 3), lr = lane & 3;
  const int tp0 = wp * 8 + lp * 4;                      // 4 consecutive p
  const int tq0 = wq * 8 + lq * 2;                      // 2 consecutive q
  const int cq = tq0 >> 1;                              // 16-byte chunk of (.., tq0) in a 16-wide row
  // r: this thread owns r = wr*16 + {2 lr, 2 lr + 1, 2 lr + 8, 2 lr + 9}  -> block wr, chunks lr and lr + 4

  const int my_items = p.n_items > (int)blockIdx.x ? (p.n_items - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;
  const int nS = (p.nI + TP_IC - 1) / TP_IC;            // stages per work item
  const int total = my_items * nS;                      // < 2^31 (checked by the launcher)

  if (tid == 0) {
    for (int s = 0; s < TP_STAGES; s++) { mbar_init(bar_full + 8 * s, 1); mbar_init(bar_empty + 8 * s, 8); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  // ---- producer (thread 0 only): flat fill index pj = (item pk of this CTA, stage pS of the item) ------------------------
  // (its counters live in shared memory: the compute loop needs every register of the 255-register budget)
  __shared__ int prod[3];
  if (tid == 0) { prod[0] = 0; prod[1] = 0; prod[2] = 0; }
  auto fill = [&]() {
    int pj = prod[0], pk = prod[1], pS = prod[2];
    if (pj >= total) return;
    const TripleItem it = p.items[blockIdx.x + (long long)pk * gridDim.x];
    const int s = pj % TP_STAGES, f = pj / TP_STAGES, I = pS * TP_IC;
    if (f > 0) mbar_wait(bar_empty + 8 * s, (uint32_t)((f - 1) & 1));
    const uint32_t dst = ring + s * TP_STAGE_BYTES, bf = bar_full + 8 * s;
    mbar_expect_tx(bf, it.diag ? 8 * TP_BLK_BYTES : 10 * TP_BLK_BYTES);
    tma_load_3d(dst + 0 * TP_BLK_BYTES, &mapE, it.q0, it.p0, I, bf);
    tma_load_3d(dst + 1 * TP_BLK_BYTES, &mapF, it.q0, it.p0, I, bf);
    tma_load_3d(dst + 2 * TP_BLK_BYTES, &mapE, it.r0, it.p0, I, bf);
    tma_load_3d(dst + 3 * TP_BLK_BYTES, &mapE, it.r0 + 16, it.p0, I, bf);
    tma_load_3d(dst + 4 * TP_BLK_BYTES, &mapF, it.r0, it.p0, I, bf);
    tma_load_3d(dst + 5 * TP_BLK_BYTES, &mapF, it.r0 + 16, it.p0, I, bf);
    tma_load_3d(dst + 6 * TP_BLK_BYTES, &mapG, it.r0, it.q0, I, bf);
    tma_load_3d(dst + 7 * TP_BLK_BYTES, &mapG, it.r0 + 16, it.q0, I, bf);
    if (!it.diag) {
      tma_load_3d(dst + 8 * TP_BLK_BYTES, &mapG, it.q0, it.r0, I, bf);          // rows r, columns q: the mirrored block
      tma_load_3d(dst + 9 * TP_BLK_BYTES, &mapG, it.q0, it.r0 + 16, I, bf);
    }
    pj++;
    if (++pS == nS) { pS = 0; pk++; }
    prod[0] = pj; prod[1] = pk; prod[2] = pS;
  };
  if (tid == 0)
    for (int n = 0; n < TP_LOOKAHEAD; n++) fill();

  // ---- per-thread shared-memory byte offsets inside a grid point's slice (swizzle: chunk ^= row & 7) -------------------
  uint32_t offPQ[4], offPR[4], offQR[2];
#pragma unroll
  for (int a = 0; a < 4; a++) {
    const int row = tp0 + a;
    offPQ[a] = row * 128 + ((cq ^ (row & 7)) << 4);
    offPR[a] = (2 + wr) * TP_BLK_BYTES + row * 128 + ((lr ^ (row & 7)) << 4);        // chunk lr; chunk lr + 4 is ^ 64
  }
#pragma unroll
  for (int b = 0; b < 2; b++) {
    const int row = tq0 + b;
    offQR[b] = (6 + wr) * TP_BLK_BYTES + row * 128 + ((lr ^ (row & 7)) << 4);
  }

  const uint32_t offT = (8 + wr) * TP_BLK_BYTES + (2 * lr) * 128 + ((cq ^ ((2 * lr) & 7)) << 4);

  const int n_gates = p.gate_every ? (p.n_items / (int)gridDim.x) / p.gate_every : 0;      // the same on every CTA
  double hqr[4][2][4], hrq[4][2][4];
  int st = 0;                 // ring stage of the current iteration
  uint32_t par = 0;           // its mbarrier phase parity
  for (int k = 0; k < my_items; k++) {
    const int diag = p.items[blockIdx.x + (long long)k * gridDim.x].diag;
#pragma unroll
    for (int a = 0; a < 4; a++)
#pragma unroll
      for (int b = 0; b < 2; b++)
#pragma unroll
        for (int c = 0; c < 4; c++) hqr[a][b][c] = hrq[a][b][c] = 0.0;

    for (int s = 0; s < nS; s++) {
      mbar_wait(bar_full + 8 * st, par);
      if (tid == 0) fill();                          // TP_LOOKAHEAD stages ahead, two iterations behind the consumers
      __syncwarp();
      const uint8_t* sl = ring_ptr + st * TP_STAGE_BYTES;
      if (diag) {
#pragma unroll 1
        for (int ii = 0; ii < TP_IC; ii++) tp_update<true>(sl + ii * TP_SLICE_BYTES, offPQ, offPR, offQR, offT, hqr, hrq);
      } else {
#pragma unroll 1
        for (int ii = 0; ii < TP_IC; ii++) tp_update<false>(sl + ii * TP_SLICE_BYTES, offPQ, offPR, offQR, offT, hqr, hrq);
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(bar_empty + 8 * st);
      if (++st == TP_STAGES) { st = 0; par ^= 1; }
    }

    // ---- write back this item's block(s) of H[p][q][r] ---------------------------------------------------------------
    // Accumulating launches (all I-chunks but the first) read the old values.  The old values of TWO p rows (32 doubles)
    // are loaded before anything of those rows is stored: with one load -> add -> store chain per 16 bytes the compiler
    // may not move a load above the preceding store, and 24 dependent round trips to L2 / HBM per work item cost 14 % of
    // a launch at BASELINE config 4 (measured: 16.3 vs 19.0 TFLOP/s with / without accumulation).
    const TripleItem cur = p.items[blockIdx.x + (long long)k * gridDim.x];
    const long long sHp = (long long)p.NPp * p.NPp;
    const int rA = cur.r0 + wr * 16 + 2 * lr;              // r = rA, rA + 1, rA + 8, rA + 9
#pragma unroll
    for (int a0 = 0; a0 < 4; a0 += 2) {
      double2 od[2][2][2], om[2][4];
#pragma unroll
      for (int aa = 0; aa < 2; aa++) {
        double* Hp = p.H + (long long)(cur.p0 + tp0 + a0 + aa) * sHp;
#pragma unroll
        for (int b = 0; b < 2; b++) {
          const double* row = Hp + (long long)(cur.q0 + tq0 + b) * p.NPp + rA;
          od[aa][b][0] = od[aa][b][1] = make_double2(0.0, 0.0);
          if (p.accumulate) { od[aa][b][0] = *reinterpret_cast<const double2*>(row); od[aa][b][1] = *reinterpret_cast<const double2*>(row + 8); }
        }
#pragma unroll
        for (int c = 0; c < 4; c++) {
          om[aa][c] = make_double2(0.0, 0.0);
          if (p.accumulate && !cur.diag)
            om[aa][c] = *reinterpret_cast<const double2*>(Hp + (long long)(rA + (c & 1) + 8 * (c >> 1)) * p.NPp + cur.q0 + tq0);
        }
      }
#pragma unroll
      for (int aa = 0; aa < 2; aa++) {
        const int a = a0 + aa;
        double* Hp = p.H + (long long)(cur.p0 + tp0 + a) * sHp;
#pragma unroll
        for (int b = 0; b < 2; b++) {
          double* row = Hp + (long long)(cur.q0 + tq0 + b) * p.NPp + rA;
          *reinterpret_cast<double2*>(row) = make_double2(hqr[a][b][0] + od[aa][b][0].x, hqr[a][b][1] + od[aa][b][0].y);
          *reinterpret_cast<double2*>(row + 8) = make_double2(hqr[a][b][2] + od[aa][b][1].x, hqr[a][b][3] + od[aa][b][1].y);
        }
        if (!cur.diag) {
#pragma unroll
          for (int c = 0; c < 4; c++) {
            double2* d = reinterpret_cast<double2*>(Hp + (long long)(rA + (c & 1) + 8 * (c >> 1)) * p.NPp + cur.q0 + tq0);
            *d = make_double2(hrq[a][0][c] + om[aa][c].x, hrq[a][1][c] + om[aa][c].y);
          }
        }
      }
    }
    // ---- gate: every CTA has at least n_gates * gate_every items, so all of them pass the same gates -----------------------
    if (n_gates && (k + 1) % p.gate_every == 0 && (k + 1) / p.gate_every <= n_gates) {
      __syncthreads();
      if (tid == 0) {
        const unsigned want = gridDim.x * (unsigned)((k + 1) / p.gate_every);
        __threadfence();
        atomicAdd(p.gate, 1u);
        unsigned seen;
        do {
          asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(p.gate) : "memory");
          if (seen < want) __nanosleep(100);
        } while (seen < want);
      }
      __syncthreads();
    }
  }
}

}  // namespace thc
