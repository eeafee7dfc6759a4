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
//   * operands are fetched by TMA (cp.async.bulk.tensor.3d, SWIZZLE_128B) as ten 16x16 FP64 blocks (2 KB each) per grid
//     point I into a TP_STAGES-deep shared-memory ring; full/empty mbarriers, no __syncthreads in the I loop.  The TMA
//     issue is done by lane 0 of warp (j mod 8) at iteration j, for iteration j + TP_STAGES - 2 (two iterations of slack
//     on the empty barrier), so the ring keeps ~120 KB in flight per SM;
//   * the 128-byte swizzle makes every 16-byte fragment load bank-conflict free (rows 4 apart differ in chunk bit 2);
//   * work items (p-tile, q-tile, r-tile) come from a host-built list ordered in groups of 8 p-tiles x 6 q-tiles x 3
//     r-tiles, so that the ~148 CTAs running at the same time share their operand tiles in L2 (5x less HBM traffic).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace thc {

constexpr int TP_PT = 16, TP_QT = 16, TP_RT = 32;
constexpr int TP_IC = 2;                                   // grid points per pipeline stage (one barrier round-trip per stage)
constexpr int TP_STAGES = 4, TP_LOOKAHEAD = TP_STAGES - 2;
constexpr int TP_BLK = 16 * 16 * 8;                        // one 16x16 FP64 block of one grid point (2 KB)
// slice of one grid point: E blocks and G blocks in 2 KB slots, F blocks in 3 KB slots with the data 512 B into the
// slot: the 128-byte swizzle is a function of the shared-memory address, so F rows land in the other 64-byte half of
// the banks than the E rows of the same (p, column) and an E/F fragment pair is read without bank conflicts
constexpr int TP_OFF_EPQ = 0, TP_OFF_EPR0 = 2048, TP_OFF_EPR1 = 4096;
constexpr int TP_OFF_GQR0 = 6144, TP_OFF_GQR1 = 8192, TP_OFF_GTQR0 = 10240, TP_OFF_GTQR1 = 12288;
constexpr int TP_OFF_FPQ = 14336 + 512, TP_OFF_FPR0 = 17408 + 512, TP_OFF_FPR1 = 20480 + 512;
constexpr int TP_SLICE_BYTES = 23552;                      // 7 x 2 KB + 3 x 3 KB
constexpr int TP_STAGE_BYTES = TP_IC * TP_SLICE_BYTES;
constexpr int TP_SMEM_BYTES = TP_STAGES * TP_STAGE_BYTES + 1024 /* alignment slack */ + 2 * TP_STAGES * 8;
constexpr int TP_THREADS = 256;

struct TripleItem { int p0, q0, r0, diag; };

struct TripleParams {
  double* H;
  const TripleItem* items;
  int n_items;
  int nI, nPp, NPp;        // padded extents: nPp % 16 == 0, NPp % 32 == 0
  int accumulate;
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


__device__ __forceinline__ double lds64(const uint8_t* base, uint32_t off) {
  return *reinterpret_cast<const double*>(base + off);
}
__device__ __forceinline__ void dmma884_tp(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

// One grid point.  The bracket s_I[p](q,r) = E_pq F_pr + F_pq E_pr is a rank-2 outer product over (q, r): one
// DMMA.8x8x4 with A = [E_pq  F_pq  0  0] (rows q) and B = [F_pr; E_pr; 0; 0] (columns r) forms it for an 8 x 8 block of
// (q, r) and leaves, in lane (g, t), s[q = pi(g)][r = 2t, 2t+1] -- next to the G values of the same (q, r), which do not
// depend on p and stay in registers for all 16 p.  Two of the four k of the DMMA are idle, which costs pipe time
// (16 clk per 64 brackets instead of 8 with DMUL + DFMA), but each lane reads 2 operand doubles per p instead of 12:
// the kernel moves from the shared-memory roof (1184 clk per grid point and CTA) to the FP64-pipe roof (768 clk).
template <bool DIAG>
__device__ __forceinline__ void tp_update(const uint8_t* sl, const uint32_t (&offA)[8], const uint32_t (&offB)[8],
                                          uint32_t offG, bool loads, double (&hq)[16][2], double (&hr)[16][2]) {
  const double2 g = lds128(sl, offG);
  double2 gt = make_double2(0.0, 0.0);
  if (!DIAG) gt = lds128(sl, offG + (TP_OFF_GTQR0 - TP_OFF_GQR0));
#pragma unroll
  for (int p = 0; p < 16; p++) {
    double a = 0.0, b = 0.0;
    if (loads) {                                    // lanes t = 0, 1 carry k = 0, 1; k = 2, 3 are zero
      a = lds64(sl, offA[p & 7] + (p >> 3) * 1024);
      b = lds64(sl, offB[p & 7] + (p >> 3) * 1024);
    }
    double s0 = 0.0, s1 = 0.0;
    dmma884_tp(s0, s1, a, b);
    hq[p][0] = fma(s0, g.x, hq[p][0]);
    hq[p][1] = fma(s1, g.y, hq[p][1]);
    if (!DIAG) {
      hr[p][0] = fma(s0, gt.x, hr[p][0]);
      hr[p][1] = fma(s1, gt.y, hr[p][1]);
    }
  }
}

// E, F: tensor maps over [nI][nPp][NPp] (innermost NPp); G, GT: over [nI][NPp][NPp] with GT_I[q][r] = G_I[r][q] (the
// mirrored block is read with the same row-q / column-r pattern as the direct one); box 16 x 16 x 1, SWIZZLE_128B.
// Grid points beyond nI (odd nI) are zero-filled by the TMA unit and add nothing.
__global__ void __launch_bounds__(TP_THREADS, 1)
triple_product_kernel(const __grid_constant__ CUtensorMap mapE, const __grid_constant__ CUtensorMap mapF,
                      const __grid_constant__ CUtensorMap mapG, const __grid_constant__ CUtensorMap mapGT,
                      const TripleParams p) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t ring = (smem_u32(smem_raw) + 1023u) & ~1023u;          // 1024-byte aligned (swizzle atom)
  const uint8_t* ring_ptr = smem_raw + (ring - smem_u32(smem_raw));
  const uint32_t bar_full = ring + TP_STAGES * TP_STAGE_BYTES;
  const uint32_t bar_empty = bar_full + TP_STAGES * 8;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, g = lane >> 2, t = lane & 3;
  const int qb = warp >> 2, rb = warp & 3;              // this warp's 8 x 8 block of the 16 q x 32 r tile, all 16 p
  const int pig = (g >> 1) + 4 * (g & 1);               // row g of the fragments <-> q = 8 qb + pi(g): rows g, g+1 differ in bit 2
  const int qrow = 8 * qb + pig;                        // q inside the tile
  const int my_items = p.n_items > (int)blockIdx.x ? (p.n_items - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;
  const int nS = (p.nI + TP_IC - 1) / TP_IC;            // stages per work item
  const int total = my_items * nS;                      // < 2^31 (checked by the launcher)

  if (tid == 0) {
    for (int s = 0; s < TP_STAGES; s++) { mbar_init(bar_full + 8 * s, 1); mbar_init(bar_empty + 8 * s, 8); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __shared__ int prod[3];                               // producer counters (thread 0): flat fill index, item, stage in item
  if (tid == 0) { prod[0] = 0; prod[1] = 0; prod[2] = 0; }
  __syncthreads();

  auto fill = [&]() {
    int pj = prod[0], pk = prod[1], pS = prod[2];
    if (pj >= total) return;
    const TripleItem it = p.items[blockIdx.x + (long long)pk * gridDim.x];
    const int s = pj % TP_STAGES, f = pj / TP_STAGES;
    if (f > 0) mbar_wait(bar_empty + 8 * s, (uint32_t)((f - 1) & 1));
    const uint32_t bf = bar_full + 8 * s;
    mbar_expect_tx(bf, TP_IC * (it.diag ? 8 : 10) * TP_BLK);
#pragma unroll
    for (int ii = 0; ii < TP_IC; ii++) {
      const uint32_t dst = ring + s * TP_STAGE_BYTES + ii * TP_SLICE_BYTES;
      const int I = pS * TP_IC + ii;
      tma_load_3d(dst + TP_OFF_EPQ, &mapE, it.q0, it.p0, I, bf);
      tma_load_3d(dst + TP_OFF_FPQ, &mapF, it.q0, it.p0, I, bf);
      tma_load_3d(dst + TP_OFF_EPR0, &mapE, it.r0, it.p0, I, bf);
      tma_load_3d(dst + TP_OFF_EPR1, &mapE, it.r0 + 16, it.p0, I, bf);
      tma_load_3d(dst + TP_OFF_FPR0, &mapF, it.r0, it.p0, I, bf);
      tma_load_3d(dst + TP_OFF_FPR1, &mapF, it.r0 + 16, it.p0, I, bf);
      tma_load_3d(dst + TP_OFF_GQR0, &mapG, it.r0, it.q0, I, bf);
      tma_load_3d(dst + TP_OFF_GQR1, &mapG, it.r0 + 16, it.q0, I, bf);
      if (!it.diag) {
        tma_load_3d(dst + TP_OFF_GTQR0, &mapGT, it.r0, it.q0, I, bf);
        tma_load_3d(dst + TP_OFF_GTQR1, &mapGT, it.r0 + 16, it.q0, I, bf);
      }
    }
    pj++;
    if (++pS == nS) { pS = 0; pk++; }
    prod[0] = pj; prod[1] = pk; prod[2] = pS;
  };
  if (tid == 0)
    for (int n = 0; n < TP_LOOKAHEAD; n++) fill();

  // ---- per-lane shared-memory byte offsets inside a grid point's slice (128-byte swizzle: chunk ^= address row & 7) ------
  // A fragment (rows q): lanes t = 0 read E[p][q], t = 1 read F[p][q];  B fragment (columns r): t = 0 F[p][r], t = 1 E[p][r]
  uint32_t offA[8], offB[8];
  {
    const int colA = qrow, colB = 8 * (rb & 1) + g;
    const bool fA = (t == 1), fB = (t == 0);            // which of the two reads the F block
#pragma unroll
    for (int k = 0; k < 8; k++) {
      offA[k] = (fA ? TP_OFF_FPQ : TP_OFF_EPQ) + k * 128 + ((((colA >> 1) ^ k ^ (fA ? 4 : 0)) << 4) | ((colA & 1) << 3));
      offB[k] = (fB ? TP_OFF_FPR0 + (rb >> 1) * 3072 : TP_OFF_EPR0 + (rb >> 1) * 2048) + k * 128 +
                ((((colB >> 1) ^ k ^ (fB ? 4 : 0)) << 4) | ((colB & 1) << 3));
    }
  }
  const uint32_t offG = TP_OFF_GQR0 + (rb >> 1) * 2048 + qrow * 128 + (((4 * (rb & 1) + t) ^ (qrow & 7)) << 4);
  const bool loads = t < 2;

  double hq[16][2], hr[16][2];     // hq[p][e] -> H[p][q][r + e],  hr[p][e] -> H[p][r + e][q],  r = 8 rb + 2t
  int st = 0;                 // ring stage of the current iteration
  uint32_t par = 0;           // its mbarrier phase parity
  for (int k = 0; k < my_items; k++) {
    const int diag = p.items[blockIdx.x + (long long)k * gridDim.x].diag;
#pragma unroll
    for (int pp = 0; pp < 16; pp++) hq[pp][0] = hq[pp][1] = hr[pp][0] = hr[pp][1] = 0.0;

    for (int s = 0; s < nS; s++) {
      mbar_wait(bar_full + 8 * st, par);
      if (tid == 0) fill();                          // TP_LOOKAHEAD stages ahead, two iterations behind the consumers
      __syncwarp();
      const uint8_t* sl = ring_ptr + st * TP_STAGE_BYTES;
      if (diag) {
#pragma unroll 1
        for (int ii = 0; ii < TP_IC; ii++) tp_update<true>(sl + ii * TP_SLICE_BYTES, offA, offB, offG, loads, hq, hr);
      } else {
#pragma unroll 1
        for (int ii = 0; ii < TP_IC; ii++) tp_update<false>(sl + ii * TP_SLICE_BYTES, offA, offB, offG, loads, hq, hr);
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(bar_empty + 8 * st);
      if (++st == TP_STAGES) { st = 0; par ^= 1; }
    }

    // ---- write back this item's block(s) of H[p][q][r] ---------------------------------------------------------------
    const TripleItem cur = p.items[blockIdx.x + (long long)k * gridDim.x];
    const long long sHp = (long long)p.NPp * p.NPp;
    const int q = cur.q0 + qrow, r = cur.r0 + 8 * rb + 2 * t;
#pragma unroll
    for (int pp = 0; pp < 16; pp++) {
      double* Hp = p.H + (long long)(cur.p0 + pp) * sHp;
      double2* d = reinterpret_cast<double2*>(Hp + (long long)q * p.NPp + r);
      double2 v = make_double2(hq[pp][0], hq[pp][1]);
      if (p.accumulate) { const double2 o = *d; v.x += o.x; v.y += o.y; }
      *d = v;
      if (!cur.diag) {
        double* m0 = Hp + (long long)r * p.NPp + q;
        double* m1 = m0 + p.NPp;
        double w0 = hr[pp][0], w1 = hr[pp][1];
        if (p.accumulate) { w0 += *m0; w1 += *m1; }
        *m0 = w0; *m1 = w1;
      }
    }
  }
}

}  // namespace thc
