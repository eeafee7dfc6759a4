// Host-side plumbing of the library: handle, bump-allocated workspace, launch helpers.
// Every launch goes through Ctx so that (a) the same code path can be run "dry" to size the workspace,
// (b) launches are counted (thc_kernel_launches) and (c) the first CUDA error is latched.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <algorithm>
#include <cstdlib>
#include <cmath>
#include <string>
#include <vector>
#include "../../include/thc.h"
#include "thc_gemm.cuh"
#include "thc_kernels.cuh"
#include "thc_triple.cuh"
#include "thc_gemm_tma.cuh"
#include "thc_ring.cuh"
#include "thc_probe.cuh"

struct thc_handle {
  int64_t o, v, NL, NP, NX;
  int64_t bL, bP7, bX, bI;           // block sizes in use
  int32_t term_mask;
  int device, sms;
  cudaStream_t stream;
  void* ws;                          // workspace base (caller's or ours)
  int64_t ws_bytes;                  // size of ws
  bool ws_owned;
  int64_t need_bytes;                // what the plan needs with the current block sizes
  int64_t launches;
  int last_cuda;
  bool smem_configured;              // triple_product_kernel opted in to its dynamic shared memory on this handle's device
  uint64_t gemm_smem_mask, ring_smem_mask;   // same, one bit per dgemm_kernel / ring_fused_kernel instantiation
  double tma_min_flop;               // GEMMs of at least this many flop may use the TMA-fed kernel (< 0: never)
  int32_t check_symmetry;
  int32_t t2sq_algorithm;            // 4 or 5 (resolved in thc_setup)
  // Alg.6 line 11: work-item lists (device memory owned by the handle), one per (nPp, NPp) shape seen
  struct TripleList { int64_t nPp, NPp; thc::TripleItem* dev; int n; };
  std::vector<TripleList> tp_lists;
  bool tp_gate = true;               // gate the long line-11 launches; cleared for good if a cooperative launch is refused
  void* encode_tiled;                // cuTensorMapEncodeTiled, resolved through the runtime (no -lcuda link)
  // B_vv streaming (THC_BVV_HOST): copy stream and double-buffer events, created on first use
  int bvv_mode;
  cudaStream_t copy_stream;
  cudaEvent_t ev_loaded[2], ev_free[2], ev_start;
  bool copy_ready;
  // per-class kernel timing (thc_profile_begin / thc_profile_end): CUDA events recorded on `stream` around every
  // launch of a class whose bit is set in prof_mask
  int prof_mask;
  std::vector<cudaEvent_t> prof_events;     // pool; pairs (start, stop)
  std::vector<int> prof_class;              // class of pair k
  std::vector<std::string> prof_desc;       // what pair k timed (printed by thc_profile_end when THC_TRACE is set)
  std::vector<double> prof_flops;          // flop (classes 0, 1) or algorithmic HBM bytes (class 2) of pair k
  std::vector<float> prof_ms;               // device time of pair k, filled by thc_profile_end
  size_t prof_done;                         // records readable through thc_profile_launch
  double prof_work[3];                      // summed over the launches of the last thc_profile_end
  size_t prof_used;                         // pairs in use
  double* sym_scratch;                      // check_symmetry: 8 doubles of device memory owned by the handle
  // CUDA graphs for launch-bound shapes (thc_options.use_graph): one cached executable graph per entry point (0 = residual,
  // 1 = energy), valid while every pointer of the call, the workspace and the stream stay the same.  The first call
  // with a new key runs eagerly (it also does the one-time opt-ins and work-list uploads), the second one is captured on
  // cap_stream (the caller's stream may be the legacy default stream, which cannot be captured) and launched, later ones
  // only launch.
  struct GraphSlot { std::vector<uintptr_t> key; int seen = 0; cudaGraphExec_t exec = nullptr; int64_t launches = 0; };
  GraphSlot graph[2];
  bool graph_on;
  cudaStream_t cap_stream;
};

namespace thc {

// Bump allocator over the workspace.  In dry mode it only tracks the high-water mark.
struct Arena {
  char* base = nullptr;
  int64_t cap = 0, top = 0, peak = 0;
  bool dry = true, overflow = false;
  double* alloc(i64 n_doubles) {
    i64 bytes = (n_doubles * 8 + 255) / 256 * 256;
    i64 at = top;
    top += bytes;
    peak = std::max(peak, top);
    if (!dry && top > cap) overflow = true;
    return reinterpret_cast<double*>(base + at);
  }
  i64 mark() const { return top; }
  void release(i64 m) { top = m; }
};

struct Gemm {
  int M, N, K;
  const double* A; i64 lda; bool akm;
  const double* B; i64 ldb; bool bkm;
  double* C; i64 ldc;
  int nbatch = 1; i64 sAb = 0, sBb = 0, sCb = 0;
  int nkb = 1; i64 sAk = 0, sBk = 0;
  double alpha_ = 1.0, beta_ = 0.0;
  const double* aux_ = nullptr; i64 ldaux = 0, sAuxb = 0;
  double* ct_ = nullptr; i64 ldct = 0, sCtb = 0;
  bool upper_ = false;
  // A(m,k): am == 'K' -> A[m*lda + k], 'M' -> A[k*lda + m].  B(n,k): bm == 'K' -> B[n*ldb + k], 'N' -> B[k*ldb + n].
  Gemm(const double* A_, i64 lda_, char am, const double* B_, i64 ldb_, char bm, double* C_, i64 ldc_, i64 M_, i64 N_, i64 K_)
      : M((int)M_), N((int)N_), K((int)K_), A(A_), lda(lda_), akm(am == 'K'), B(B_), ldb(ldb_), bkm(bm == 'K'), C(C_), ldc(ldc_) {}
  Gemm& batch(i64 n, i64 sa, i64 sb, i64 sc) { nbatch = (int)n; sAb = sa; sBb = sb; sCb = sc; return *this; }
  Gemm& kbatch(i64 n, i64 sa, i64 sb) { nkb = (int)n; sAk = sa; sBk = sb; return *this; }
  Gemm& ab(double a, double b) { alpha_ = a; beta_ = b; return *this; }
  Gemm& aux(const double* p, i64 ld, i64 sb) { aux_ = p; ldaux = ld; sAuxb = sb; return *this; }
  Gemm& transposed_copy(double* p, i64 ld, i64 sb) { ct_ = p; ldct = ld; sCtb = sb; return *this; }   // Ct_b[n][m] too
  Gemm& upper_only() { upper_ = true; return *this; }    // symmetric M x M product: tiles strictly below the diagonal are skipped
};

// tile configurations of dgemm_kernel
#ifndef THC_BIG_BK
#define THC_BIG_BK 16
#define THC_BIG_ST 4
#endif
#define THC_BIG 128, 128, THC_BIG_BK, 2, 4, THC_BIG_ST
#define THC_MID 128, 64, 16, 4, 2, 4
#define THC_SMALL 64, 64, 16, 2, 2, 4
#define THC_TINYK 64, 64, 16, 2, 2, 2      // K <= 32: the whole K in the two stages, six CTAs per SM hide each other's latency
constexpr int BIG_THREADS = 256, SMALL_THREADS = 128;
constexpr int gemm_smem_bytes(int BM, int BN, int BK, int ST, bool akm, bool bkm) {
  return ST * ((akm ? BM * BK : BK * (BM + 2)) + (bkm ? BN * BK : BK * (BN + 2))) * 8;
}
#define THC_TALL 160, 64, 16, 4, 2, 4       // extents just above 128 (o = 150 at BASELINE config 3): one 160-wide tile instead
#define THC_WIDE 64, 160, 16, 2, 4, 4       // of two 128-wide ones; K-major, 16-byte aligned operands only
// tile 0: 128x128 (one CTA per SM), 1: 128x64 (two), 2: 64x64 (three), 3: 64x64 with a 2-stage ring for K <= 32 (six),
// 4: 160x64, 5: 64x160 (one)
struct TileCfg { int BM, BN, per_sm; double lone_rate, pipe_share; };
constexpr TileCfg TILE_CFGS[6] = {{128, 128, 1, 1.0, 1.0}, {128, 64, 2, 0.7, 0.9}, {64, 64, 3, 0.5, 0.75}, {64, 64, 6, 0.5, 0.75},
                                  {160, 64, 1, 0.85, 0.85}, {64, 160, 1, 0.85, 0.85}};

// The opt-in to more than 48 KB of dynamic shared memory is a per-device attribute of the kernel: it is recorded per
// handle (one handle = one device), bit `bit` of `mask`, never per process.
template <typename K>
static cudaError_t opt_in_smem(K k, int bytes, uint64_t& mask, int bit) {
  if (mask & (1ull << bit)) return cudaSuccess;
  cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
  if (e == cudaSuccess) mask |= 1ull << bit;
  return e;
}

template <bool AKM, bool BKM, bool AL16>
static cudaError_t launch_gemm_variant(int tile, dim3 grid, cudaStream_t st, const GemmParams& p, uint64_t& mask) {
  const int bit = tile * 8 + (AKM ? 4 : 0) + (BKM ? 2 : 0) + (AL16 ? 1 : 0);
  cudaError_t e = cudaSuccess;
  if (tile >= 4) {                          // only instantiated for K-major, aligned operands (the caller checks)
    if (!(AKM && BKM && AL16)) return cudaErrorInvalidValue;
    const int sm = gemm_smem_bytes(160, 64, 16, 4, true, true);
    if (tile == 4) {
      auto k = dgemm_kernel<THC_TALL, true, true, true>;
      if ((e = opt_in_smem(k, sm, mask, 32)) != cudaSuccess) return e;
      k<<<grid, BIG_THREADS, sm, st>>>(p);
    } else {
      auto k = dgemm_kernel<THC_WIDE, true, true, true>;
      if ((e = opt_in_smem(k, sm, mask, 33)) != cudaSuccess) return e;
      k<<<grid, BIG_THREADS, sm, st>>>(p);
    }
    return cudaPeekAtLastError();
  }
  if (tile == 0) {
    auto k = dgemm_kernel<THC_BIG, AKM, BKM, AL16>;
    int sm = gemm_smem_bytes(128, 128, THC_BIG_BK, THC_BIG_ST, AKM, BKM);
    if ((e = opt_in_smem(k, sm, mask, bit)) != cudaSuccess) return e;
    k<<<grid, BIG_THREADS, sm, st>>>(p);
  } else if (tile == 1) {
    auto k = dgemm_kernel<THC_MID, AKM, BKM, AL16>;
    int sm = gemm_smem_bytes(128, 64, 16, 4, AKM, BKM);
    if ((e = opt_in_smem(k, sm, mask, bit)) != cudaSuccess) return e;
    k<<<grid, BIG_THREADS, sm, st>>>(p);
  } else if (tile == 2) {
    auto k = dgemm_kernel<THC_SMALL, AKM, BKM, AL16>;
    int sm = gemm_smem_bytes(64, 64, 16, 4, AKM, BKM);
    if ((e = opt_in_smem(k, sm, mask, bit)) != cudaSuccess) return e;
    k<<<grid, SMALL_THREADS, sm, st>>>(p);
  } else {
    auto k = dgemm_kernel<THC_TINYK, AKM, BKM, AL16>;
    int sm = gemm_smem_bytes(64, 64, 16, 2, AKM, BKM);
    k<<<grid, SMALL_THREADS, sm, st>>>(p);         // 32 KB of shared memory: no opt-in needed
  }
  return cudaPeekAtLastError();
}

struct Ctx {
  thc_handle* h;
  Arena ar;
  bool dry;
  int status = THC_OK;
  i64 splitk_need = 0;          // doubles of split-K scratch the plan needs (dry) ...
  double* splitk = nullptr;     // ... and the buffer (real run)
  i64 splitk_cap = 0;

  bool ok() const { return status == THC_OK; }
  void check(cudaError_t e) {
    if (e != cudaSuccess && status == THC_OK) { status = THC_ERR_CUDA; h->last_cuda = (int)e; }
  }
  void launched() { h->launches++; check(cudaPeekAtLastError()); }
  // kernel classes for thc_profile_*: 0 = DMMA GEMM (+ its split-K reduce), 1 = Alg.6 line 11, 2 = Hadamard / reduction
  void prof_start(int cls, const char* desc = "", double flops = 0.0) {
    if (!(h->prof_mask & (1 << cls))) return;
    if (h->prof_used * 2 + 2 > h->prof_events.size()) {
      cudaEvent_t a, b;
      if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) { check(cudaGetLastError()); return; }
      h->prof_events.push_back(a); h->prof_events.push_back(b);
      h->prof_class.push_back(cls);
      h->prof_desc.emplace_back();
      h->prof_flops.push_back(0.0);
    }
    h->prof_class[h->prof_used] = cls;
    h->prof_desc[h->prof_used] = desc;
    h->prof_flops[h->prof_used] = flops;
    cudaEventRecord(h->prof_events[h->prof_used * 2], h->stream);
  }
  void prof_stop(int cls) {
    if (!(h->prof_mask & (1 << cls))) return;
    if (h->prof_used * 2 + 2 > h->prof_events.size()) return;
    cudaEventRecord(h->prof_events[h->prof_used * 2 + 1], h->stream);
    h->prof_used++;
  }
  int ew_blocks(i64 n, int per = 256) const { return (int)std::max<i64>(1, std::min<i64>((n + per - 1) / per, (i64)h->sms * 16)); }

  // ---- GEMM ----------------------------------------------------------------------------------------------------
  typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                               const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                               CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  EncodeFn encode_fn() {
    if (!h->encode_tiled) {
      void* fn = nullptr;
      cudaDriverEntryPointQueryResult q;
      if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) != cudaSuccess || !fn) return nullptr;
      h->encode_tiled = fn;
    }
    return reinterpret_cast<EncodeFn>(h->encode_tiled);
  }
  // TMA descriptor of a K-major GEMM operand: element (k, row, kb, b) at base[row * ld + k + kb * sk + b * sb]; box = 8 k x
  // box_rows rows (64-byte rows, no swizzle: the [k/8][row][8] shared-memory layout).  A zero stride (broadcast operand,
  // single k-batch) becomes a dimension of extent 1.  Returns false when the driver rejects the layout.
  bool make_map4(CUtensorMap* m, const double* base, i64 K, i64 rows, i64 ld, i64 nkb, i64 sk, i64 nb, i64 sb, int box_rows) {
    EncodeFn enc = encode_fn();
    if (!enc) return false;
    if (sk == 0) nkb = 1;
    if (sb == 0) nb = 1;
    const cuuint64_t dims[4] = {(cuuint64_t)K, (cuuint64_t)rows, (cuuint64_t)nkb, (cuuint64_t)nb};
    const cuuint64_t dflt = (cuuint64_t)ld * 8;
    const cuuint64_t strides[3] = {(cuuint64_t)ld * 8, sk ? (cuuint64_t)sk * 8 : dflt, sb ? (cuuint64_t)sb * 8 : dflt};
    const cuuint32_t box[4] = {8, (cuuint32_t)box_rows, 1, 1}, es[4] = {1, 1, 1, 1};
    CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, const_cast<double*>(base), dims, strides, box, es,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
  }
  // TMA-fed persistent kernel (thc_gemm_tma.cuh) for tiles 0 (128x128), 4 (160x64), 5 (64x160).  false -> not launched
  // (the caller falls back to the cp.async kernel).
  template <int BM, int BN, int WM, int WN, int ST>
  bool launch_tma_cfg(const GemmParams& p, const CUtensorMap& mA, const CUtensorMap& mB, int bit) {
    auto k = dgemm_tma_kernel<BM, BN, WM, WN, ST>;
    const int sm = tg_smem_bytes(BM, BN, ST);
    if (opt_in_smem(k, sm, h->gemm_smem_mask, bit) != cudaSuccess) { cudaGetLastError(); return false; }
    const i64 tm = (p.M + BM - 1) / BM, tn = (p.N + BN - 1) / BN;
    const i64 tiles = (p.upper_only ? tm * (tm + 1) / 2 : tm * tn) * p.splits * p.batch;
    const int grid = (int)std::min<i64>(tiles, h->sms);
    k<<<grid, TG_THREADS, sm, h->stream>>>(mA, mB, p);
    return true;
  }
  bool launch_tma(int tile, const Gemm& g, const GemmParams& p) {
    if (!(tile == 0 || tile == 4 || tile == 5) || !g.akm || !g.bkm) return false;
    if (g.upper_ && (tile != 0 || g.M != g.N)) return false;
    const int BM = TILE_CFGS[tile].BM, BN = TILE_CFGS[tile].BN;
    CUtensorMap mA, mB;
    if (!make_map4(&mA, g.A, g.K, g.M, g.lda, g.nkb, g.sAk, g.nbatch, g.sAb, BM) ||
        !make_map4(&mB, g.B, g.K, g.N, g.ldb, g.nkb, g.sBk, g.nbatch, g.sBb, BN)) return false;
    if (tile == 0) return launch_tma_cfg<128, 128, 2, 4, 6>(p, mA, mB, 40);
    if (tile == 4) return launch_tma_cfg<160, 64, 4, 2, 6>(p, mA, mB, 41);
    return launch_tma_cfg<64, 160, 2, 4, 6>(p, mA, mB, 42);
  }

  void gemm(const Gemm& g) {
    if (g.M <= 0 || g.N <= 0 || g.nbatch <= 0) return;
    // Tile shape and split-K factor: minimise  waves x (k-iterations per CTA + fixed cost) x tile area / tile rate  over
    // TILE_CFGS x splits; a split-K pass adds a partial-tile write and a reduction.
    const i64 kiters = (i64)g.nkb * ((g.K + 15) / 16);
    auto even = [](i64 x) { return (x & 1) == 0; };
    const bool al16 = ((reinterpret_cast<uintptr_t>(g.A) | reinterpret_cast<uintptr_t>(g.B)) & 15) == 0 && even(g.lda) &&
                      even(g.ldb) && even(g.sAb) && even(g.sBb) && even(g.sAk) && even(g.sBk);
    int tile = 2, splits = 1; double best = 1e300;
    for (int cfg = 0; cfg < 6; cfg++) {
      if (cfg == 3) continue;
      const TileCfg& tc = TILE_CFGS[cfg];
      if (cfg < 2 && (g.M <= 64 || g.N <= (cfg == 0 ? 64 : 32))) continue;
      // 160-wide tiles: only where they save a whole row / column of 128-tiles, K-major aligned operands, plain epilogue
      if (cfg == 4 && !(g.akm && g.bkm && al16 && !g.upper_ && g.M > 128 && (g.M + 159) / 160 * 160 < (g.M + 127) / 128 * 128)) continue;
      if (cfg == 5 && !(g.akm && g.bkm && al16 && !g.upper_ && g.N > 128 && (g.N + 159) / 160 * 160 < (g.N + 127) / 128 * 128)) continue;
      i64 tmn = (i64)((g.M + tc.BM - 1) / tc.BM) * ((g.N + tc.BN - 1) / tc.BN) * g.nbatch;
      if (g.upper_) {                                       // only tiles that reach the diagonal or lie above it work
        tmn = 0;
        for (i64 tm = 0; tm * tc.BM < g.M; tm++)
          for (i64 tn = 0; tn * tc.BN < g.N; tn++) tmn += ((tn + 1) * tc.BN > tm * tc.BM);
        tmn *= g.nbatch;
      }
      const double slots = (double)h->sms * tc.per_sm;
      const int smax = g.ct_ ? 1 : (int)std::max<i64>(1, std::min<i64>(64, kiters / 8));   // the transposed copy is written by the main kernel only
      for (int sp = 1; sp <= smax; sp++) {
        const double waves = std::ceil((double)tmn * sp / slots);
        // per-CTA DMMA rate relative to a 128x128 CTA that owns an SM: a lone smaller CTA cannot fill the pipe
        // (lone_rate), several of them share pipe_share of it
        const double conc = std::min((double)tc.per_sm, std::ceil((double)tmn * sp / h->sms));
        const double rate = std::min(tc.lone_rate, tc.pipe_share / conc);
        double t = waves * ((double)kiters / sp + 6.0) * tc.BM * tc.BN / rate;
        if (sp > 1) t += 0.025 * sp * (double)g.M * g.N * g.nbatch;     // partial-tile write + reduction at ~5 TB/s, same units
        if (t < best * (sp > 1 ? 0.97 : 1.0)) { best = t; tile = cfg; splits = sp; }
      }
    }
    if (tile == 2 && kiters <= 2 && splits == 1) tile = 3;      // tiny K: latency-bound CTAs, run six per SM
    const TileCfg& tc = TILE_CFGS[tile];
    const i64 tiles_mn = (i64)((g.M + tc.BM - 1) / tc.BM) * ((g.N + tc.BN - 1) / tc.BN);
    const i64 per = (i64)g.nbatch * g.M * g.N;
    if (splits > 1) splitk_need = std::max(splitk_need, per * splits);
    if (dry || !ok()) return;
    // The scratch was sized by a dry run of the unsharded plan; a shard (other nl / row counts) may prefer more splits
    // than it has room for: take the largest split factor that fits instead of failing.
    if (splits > 1 && per * splits > splitk_cap) splits = (int)std::max<i64>(1, splitk_cap / per);
    // grid.z carries batch x splits and is limited to 65535: long batches go out as several launches
    if ((i64)g.nbatch * splits > 65535) {
      const int chunk = std::max(1, 65535 / splits);
      for (int b0 = 0; b0 < g.nbatch && ok(); b0 += chunk) {
        Gemm part = g;
        part.nbatch = std::min(chunk, g.nbatch - b0);
        part.A = g.A + (i64)b0 * g.sAb; part.B = g.B + (i64)b0 * g.sBb; part.C = g.C + (i64)b0 * g.sCb;
        if (g.aux_) part.aux_ = g.aux_ + (i64)b0 * g.sAuxb;
        if (g.ct_) part.ct_ = g.ct_ + (i64)b0 * g.sCtb;
        gemm(part);
      }
      return;
    }

    GemmParams p;
    p.A = g.A; p.B = g.B; p.aux = g.aux_;
    p.M = g.M; p.N = g.N; p.K = g.K;
    p.lda = g.lda; p.ldb = g.ldb; p.ldaux = g.ldaux;
    p.batch = g.nbatch; p.sAb = g.sAb; p.sBb = g.sBb; p.sAuxb = g.sAuxb;
    p.kbatch = g.nkb; p.sAk = g.sAk; p.sBk = g.sBk;
    p.splits = splits; p.alpha = g.alpha_; p.beta = g.beta_;
    p.Ct = g.ct_; p.ldct = g.ldct; p.sCtb = g.sCtb;
    p.upper_only = g.upper_ ? 1 : 0;
    if (splits > 1) { p.C = splitk; p.ldc = g.N; p.sCb = (i64)g.M * g.N; p.sCs = per; }
    else            { p.C = g.C; p.ldc = g.ldc; p.sCb = g.sCb; p.sCs = 0; }

    dim3 grid((unsigned)tiles_mn, 1, (unsigned)((i64)g.nbatch * splits));
    cudaError_t e;
    char desc[160];
    if (h->prof_mask & 1)
      snprintf(desc, sizeof desc, "gemm %s M=%d N=%d K=%d batch=%d kbatch=%d splits=%d %c%c%s", tile == 0 ? "big" : (tile == 1 ? "mid" : (tile == 2 ? "small" : (tile == 3 ? "tinyK" : (tile == 4 ? "tall" : "wide")))), g.M, g.N, g.K,
               g.nbatch, g.nkb, splits, g.akm ? 'K' : 'M', g.bkm ? 'K' : 'N', al16 ? "" : " unaligned");
    prof_start(0, desc, 2.0 * g.M * g.N * (double)g.K * g.nbatch * g.nkb * (g.upper_ ? 0.5 * (1.0 + (double)tc.BN / g.N) : 1.0));
    const int sel = (g.akm ? 4 : 0) | (g.bkm ? 2 : 0) | (al16 ? 1 : 0);
    // large aligned K-major products go to the TMA-fed persistent kernel; small ones (launch-bound shapes, where encoding
    // two descriptors costs more than it saves) and everything else to the cp.async kernel
    const bool want_tma = al16 && h->tma_min_flop >= 0 && 2.0 * g.M * g.N * (double)g.K * g.nbatch * g.nkb >= h->tma_min_flop;
    if (want_tma && launch_tma(tile, g, p)) {
      e = cudaPeekAtLastError();
    } else
    switch (sel) {
      case 7: e = launch_gemm_variant<true, true, true>(tile, grid, h->stream, p, h->gemm_smem_mask); break;
      case 6: e = launch_gemm_variant<true, true, false>(tile, grid, h->stream, p, h->gemm_smem_mask); break;
      case 5: e = launch_gemm_variant<true, false, true>(tile, grid, h->stream, p, h->gemm_smem_mask); break;
      case 4: e = launch_gemm_variant<true, false, false>(tile, grid, h->stream, p, h->gemm_smem_mask); break;
      case 3: e = launch_gemm_variant<false, true, true>(tile, grid, h->stream, p, h->gemm_smem_mask); break;
      case 2: e = launch_gemm_variant<false, true, false>(tile, grid, h->stream, p, h->gemm_smem_mask); break;
      case 1: e = launch_gemm_variant<false, false, true>(tile, grid, h->stream, p, h->gemm_smem_mask); break;
      default: e = launch_gemm_variant<false, false, false>(tile, grid, h->stream, p, h->gemm_smem_mask); break;
    }
    h->launches++;
    check(e);
    if (splits > 1) {
      ReduceParams r;
      r.part = splitk; r.dst = g.C; r.aux = g.aux_;
      r.M = g.M; r.N = g.N; r.batch = g.nbatch; r.splits = splits;
      r.ldd = g.ldc; r.sDb = g.sCb; r.ldaux = g.ldaux; r.sAuxb = g.sAuxb;
      r.alpha = g.alpha_; r.beta = g.beta_;
      r.skip_bm = g.upper_ ? tc.BM : 0; r.skip_bn = g.upper_ ? tc.BN : 0;
      reduce_splits_kernel<<<ew_blocks(per), 256, 0, h->stream>>>(r);
      launched();
    }
    prof_stop(0);
  }

  // ---- element-wise / reduction launches -------------------------------------------------------------------------
// `bytes` = algorithmic HBM bytes of the launch (every operand element read once, every result written once)
#define THC_EW(kernel, n, bytes, ...)                                   \
  do {                                                                  \
    if (dry || !ok()) return;                                           \
    prof_start(2, #kernel, (double)(bytes));                            \
    kernel<<<ew_blocks(n), 256, 0, h->stream>>>(__VA_ARGS__);           \
    launched();                                                         \
    prof_stop(2);                                                       \
  } while (0)

  void transpose(const double* in, double* out, i64 rows, i64 cols) {
    if (dry || !ok()) return;
    dim3 grid((unsigned)((cols + 31) / 32), (unsigned)((rows + 31) / 32)), blk(32, 8);
    prof_start(2, "transpose_kernel", 16.0 * rows * cols);
    transpose_kernel<<<grid, blk, 0, h->stream>>>(in, out, (int)rows, (int)cols);
    launched();
    prof_stop(2);
  }
  void fill(double* x, i64 n, double val) { THC_EW(fill_kernel, n, 8.0 * n, x, n, val); }
  void hadamard(const double* a, const double* b, double* out, i64 n) { THC_EW(hadamard_kernel, n, 24.0 * n, a, b, out, n); }
  void axpby(const double* a, const double* b, double ca, double cb, double* out, i64 n) {
    THC_EW(axpby_kernel, n, 24.0 * n, a, b, ca, cb, out, n);
  }
  void had2_diff(const double* a, const double* b, const double* c, const double* d, double* out, i64 n) {
    THC_EW(had2_diff_kernel, n, 40.0 * n, a, b, c, d, out, n);
  }
  void combine(double* Mo, const double* Mv, const double* omat, const double* vmat, double* C3, i64 np2, i64 nl) {
    THC_EW(combine_kernel, np2, 8.0 * np2 * (3.0 * nl + 4.0), Mo, Mv, omat, vmat, C3, np2, (int)nl);
  }
  void rowdot(const double* X, i64 ldx, const double* T, i64 sTb, i64 ldT, double* out, i64 ldo, i64 nb, i64 nr, i64 n) {
    THC_EW(rowdot_kernel, nb * nr * 8 /* eight lanes per row */, 8.0 * ((double)nb * nr * n + (double)nr * n + (double)nb * nr), X, ldx, T, sTb, ldT, out, ldo, (int)nb, (int)nr, (int)n);
  }
  void coldot(const double* X, i64 ldx, const double* T, i64 sTb, i64 ldT, double* out, i64 ldo, i64 nb, i64 nc, i64 n) {
    THC_EW(coldot_kernel, nb * nc, 8.0 * ((double)nb * nc * n + (double)nc * n + (double)nb * nc), X, ldx, T, sTb, ldT, out, ldo, (int)nb, (int)nc, (int)n);
  }
  void rowscale(const double* X, i64 ldx, const double* Mrow, i64 ldm, const double* add, double alpha, double* out,
                i64 nb, i64 n, i64 nc) {
    const double bytes = 8.0 * ((double)nb * n * nc * (add ? 2.0 : 1.0) + (double)n * nc + (double)nb * nc);
    const bool vec = ((nc | ldx | ldm) & 1) == 0 &&
                     ((reinterpret_cast<uintptr_t>(X) | reinterpret_cast<uintptr_t>(Mrow) | reinterpret_cast<uintptr_t>(add) |
                       reinterpret_cast<uintptr_t>(out)) & 15) == 0;
    if (vec) THC_EW(rowscale2_kernel, nb * n * nc / 2, bytes, X, ldx, Mrow, ldm, add, alpha, out, (int)nb, (int)n, (int)nc);
    else THC_EW(rowscale_kernel, nb * n * nc, bytes, X, ldx, Mrow, ldm, add, alpha, out, (int)nb, (int)n, (int)nc);
  }
  void rowscale_inplace(double* T, const double* Mrow, i64 ldm, double alpha, i64 nb, i64 n, i64 nc) {
    THC_EW(rowscale_inplace_kernel, nb * n * nc, 8.0 * (2.0 * nb * n * nc + (double)nb * nc), T, Mrow, ldm, alpha, (int)nb, (int)n, (int)nc);
  }
  void qm(double* G1, const double* Xo, const double* ZA, i64 o, i64 nl, i64 NP) {
    THC_EW(qm_kernel, o * nl * NP, 8.0 * (2.0 * o * nl * NP + (double)o * NP + (double)nl * NP), G1, Xo, ZA, (int)o, (int)nl, (int)NP);
  }
  void symmetrize(const double* P, double* out, i64 n, double scale) {
    if (dry || !ok()) return;
    dim3 grid((unsigned)((n + 31) / 32), (unsigned)((n + 31) / 32)), blk(32, 8);
    prof_start(2, "symmetrize_kernel", 16.0 * n * n);
    symmetrize_kernel<<<grid, blk, 0, h->stream>>>(P, out, (int)n, scale);
    launched();
    prof_stop(2);
  }
  void mirror_upper(double* A, i64 n, i64 nbatch = 1) {     // nbatch matrices n x n, densely packed
    if (dry || !ok()) return;
    dim3 grid((unsigned)((n + 31) / 32), (unsigned)((n + 31) / 32), (unsigned)nbatch), blk(32, 8);
    prof_start(2, "mirror_upper_kernel", 8.0 * n * n * nbatch);
    mirror_upper_kernel<<<grid, blk, 0, h->stream>>>(A, (int)n);
    launched();
    prof_stop(2);
  }
  void t1_eps(const double* eps, const double* t1, double* out, i64 o, i64 v) { THC_EW(t1_eps_kernel, o * v, 24.0 * o * v, eps, t1, out, (int)o, (int)v); }
  void pair_accumulate(const double* J, const double* FA, i64 ldfa, const double* FB, i64 ldfb, double* out, i64 n, i64 n1, i64 n2) {
    THC_EW(pair_accumulate_kernel, n * n, 8.0 * n * n * (n1 * n2 + 2.0), J, FA, ldfa, FB, ldfb, out, (int)n, (int)n1, (int)n2);
  }
  void diag(const double* A, double* d, i64 n) { THC_EW(diag_kernel, n, 16.0 * n, A, d, (int)n); }
  // PCG over nrows independent systems (one warp per row)
  void pcg_init(const double* r, const double* d, double* p, double* rz, i64 nrows, i64 n) {
    THC_EW(pcg_init_kernel, nrows * 32, 8.0 * (2.0 * nrows * n + n + nrows), r, d, p, rz, (int)nrows, (int)n);
  }
  void pcg_iter(double* x, double* r, double* p, const double* Sp, const double* d, double* rz, i64 nrows, i64 n) {
    THC_EW(pcg_iter_kernel, nrows * 32, 8.0 * (7.0 * nrows * n + n + 2.0 * nrows), x, r, p, Sp, d, rz, (int)nrows, (int)n);
  }
  void copy(const double* src, double* dst, i64 n) {
    if (dry || !ok()) return;
    check(cudaMemcpyAsync(dst, src, (size_t)n * 8, cudaMemcpyDeviceToDevice, h->stream));
  }
  void fock(const double* eps, const double* xi_oo, const double* xi_vv, double* FooT, double* Fvv, i64 o, i64 v) {
    THC_EW(fock_kernel, o * o + v * v, 16.0 * (o * o + v * v), eps, xi_oo, xi_vv, FooT, Fvv, (int)o, (int)v);
  }
  void sum6(const double* const t[6], double* out, i64 n) {
    THC_EW(sum6_kernel, n, 56.0 * n, t[0], t[1], t[2], t[3], t[4], t[5], out, n);
  }
  // partial sums for the energy; `partial` must hold dot_blocks() / zee_blocks() doubles
  int dot_blocks(i64 n) const { return ew_blocks(n, 1024); }
  void dot_partial(const double* a, const double* b, i64 n, double* partial) {
    if (dry || !ok()) return;
    prof_start(2, "dot_partial_kernel", 16.0 * n);
    dot_partial_kernel<<<dot_blocks(n), 256, 0, h->stream>>>(a, b, n, partial);
    launched();
    prof_stop(2);
  }
  i64 zee_blocks(i64 NP, i64 nl) const { i64 t = (NP + 31) / 32; return t * t * nl; }
  void zee_partial(const double* Z, const double* E, i64 NP, i64 nl, double* partial) {
    if (dry || !ok()) return;
    unsigned t = (unsigned)((NP + 31) / 32);
    dim3 grid(t, t, (unsigned)nl), blk(32, 8);
    prof_start(2, "zee_partial_kernel", 8.0 * NP * NP * (nl + 1.0));
    zee_partial_kernel<<<grid, blk, 0, h->stream>>>(Z, E, (int)NP, partial);
    launched();
    prof_stop(2);
  }
  void final_sum(const double* pa, i64 na, double ca, const double* pb, i64 nb, double cb, double* out, int accumulate) {
    if (dry || !ok()) return;
    prof_start(2, "final_sum_kernel", 8.0 * (na + nb));
    final_sum_kernel<<<1, 1024, 0, h->stream>>>(pa, na, ca, pb, nb, cb, out, accumulate);
    launched();
    prof_stop(2);
  }
  // ---- Alg.7 lines 12-19 fused (o <= 64) ------------------------------------------------------------------------------
  static bool ring_supported(i64 o) { return o <= 64; }
  template <int KT>
  void ring_launch(const RingParams& p, bool al16, dim3 grid) {
    const int sm = ring_smem_bytes(KT);
    if (al16) {
      check(opt_in_smem(ring_fused_kernel<KT, true>, sm, h->ring_smem_mask, 2 * KT));
      if (ok()) ring_fused_kernel<KT, true><<<grid, RG_THREADS, sm, h->stream>>>(p);
    } else {
      check(opt_in_smem(ring_fused_kernel<KT, false>, sm, h->ring_smem_mask, 2 * KT + 1));
      if (ok()) ring_fused_kernel<KT, false><<<grid, RG_THREADS, sm, h->stream>>>(p);
    }
  }
  // FYT[b][j][I] = sum_J (sum_i YoT[I][i] RYT[b][J][i]) V[I][J] Yo[j][J]
  void ring_fused(const double* YoT, const double* RYT, const double* V, const double* Yo, double* FYT, i64 NX, i64 o, i64 npb) {
    if (dry || !ok()) return;
    RingParams p;
    p.YoT = YoT; p.RYT = RYT; p.V = V; p.Yo = Yo; p.FYT = FYT; p.NX = (int)NX; p.o = (int)o; p.npb = (int)npb;
    const bool al16 = (o % 2 == 0) && (NX % 2 == 0) &&
                      ((reinterpret_cast<uintptr_t>(RYT) | reinterpret_cast<uintptr_t>(V) | reinterpret_cast<uintptr_t>(Yo)) & 15) == 0;
    dim3 grid((unsigned)((NX + RG_BM - 1) / RG_BM), (unsigned)npb);
    char desc[96];
    if (h->prof_mask & 1) snprintf(desc, sizeof desc, "ring_fused NX=%d o=%d batch=%d", (int)NX, (int)o, (int)npb);
    prof_start(0, desc, 4.0 * o * (double)NX * NX * npb);
    switch ((o + 7) / 8) {
      case 1: ring_launch<1>(p, al16, grid); break;
      case 2: ring_launch<2>(p, al16, grid); break;
      case 3: ring_launch<3>(p, al16, grid); break;
      case 4: ring_launch<4>(p, al16, grid); break;
      case 5: ring_launch<5>(p, al16, grid); break;
      case 6: ring_launch<6>(p, al16, grid); break;
      case 7: ring_launch<7>(p, al16, grid); break;
      default: ring_launch<8>(p, al16, grid); break;
    }
    launched();
    prof_stop(0);
  }

  // ---- B_vv streaming (THC_BVV_HOST / THC_BVV_PROVIDER) ------------------------------------------------------------
  void bvv_begin() {
    if (!ok() || h->bvv_mode != THC_BVV_HOST) return;
    if (!h->copy_ready) {
      check(cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking));
      for (int k = 0; k < 2; k++) {
        check(cudaEventCreateWithFlags(&h->ev_loaded[k], cudaEventDisableTiming));
        check(cudaEventCreateWithFlags(&h->ev_free[k], cudaEventDisableTiming));
      }
      check(cudaEventCreateWithFlags(&h->ev_start, cudaEventDisableTiming));
      h->copy_ready = ok();
    }
    // the copy stream may not touch the double buffer before earlier work on the compute stream has finished with it
    check(cudaEventRecord(h->ev_start, h->stream));
    check(cudaStreamWaitEvent(h->copy_stream, h->ev_start, 0));
  }
  void bvv_copy(double* dst, const double* host, i64 L0, i64 nl, i64 v, i64 blk) {
    if (!ok()) return;
    if (blk >= 2) check(cudaStreamWaitEvent(h->copy_stream, h->ev_free[blk & 1], 0));
    check(cudaMemcpyAsync(dst, host + L0 * v * v, (size_t)(nl * v * v) * 8, cudaMemcpyHostToDevice, h->copy_stream));
    check(cudaEventRecord(h->ev_loaded[blk & 1], h->copy_stream));
  }
  void bvv_wait_loaded(i64 blk) { if (ok()) check(cudaStreamWaitEvent(h->stream, h->ev_loaded[blk & 1], 0)); }
  void bvv_release(i64 blk) { if (ok()) check(cudaEventRecord(h->ev_free[blk & 1], h->stream)); }
  void bvv_provide(const thc_bvv_provider* pr, i64 L0, i64 nl, double* dst) {
    if (!ok()) return;
    if (!pr || !pr->fill) { status = THC_ERR_INVALID_ARG; return; }
    if (pr->fill(pr->ctx, L0, nl, dst, (void*)h->stream) != 0) status = THC_ERR_PROVIDER;
  }

  // TMA descriptor over a [d2][d1][d0] FP64 array (d0 contiguous), box 16 x 16 x 1, 128-byte swizzle.
  bool make_map3(CUtensorMap* m, const double* base, i64 d0, i64 d1, i64 d2) {
    typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                 const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                 CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    if (!h->encode_tiled) {
      void* fn = nullptr;
      cudaDriverEntryPointQueryResult q;
      if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) != cudaSuccess || !fn) {
        check(cudaErrorNotSupported);
        return false;
      }
      h->encode_tiled = fn;
    }
    const cuuint64_t dims[3] = {(cuuint64_t)d0, (cuuint64_t)d1, (cuuint64_t)d2};
    const cuuint64_t strides[2] = {(cuuint64_t)d0 * 8, (cuuint64_t)d0 * (cuuint64_t)d1 * 8};
    const cuuint32_t box[3] = {16, 16, (cuuint32_t)TP_IC}, es[3] = {1, 1, 1};
    CUresult r = reinterpret_cast<EncodeFn>(h->encode_tiled)(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<double*>(base), dims,
                                                             strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                                                             CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { check(cudaErrorInvalidValue); return false; }
    return true;
  }
  // Work items of Alg.6 line 11 in an L2-friendly order: groups of 8 p-tiles x 6 q-tiles x 3 r-tiles run at the same time.
  const thc_handle::TripleList* triple_items(i64 nPp, i64 NPp) {
    for (const auto& l : h->tp_lists) if (l.nPp == nPp && l.NPp == NPp) return &l;
    std::vector<TripleItem> items;
    const int npt = (int)(nPp / TP_PT), nqb = (int)(NPp / TP_QT), nrb = (int)(NPp / TP_RT);
    for (int rb0 = 0; rb0 < nrb; rb0 += 3)
      for (int qb0 = 0; qb0 < nqb && qb0 <= 2 * std::min(rb0 + 2, nrb - 1) + 1; qb0 += 6)
        for (int pt0 = 0; pt0 < npt; pt0 += 8)
          for (int pt = pt0; pt < std::min(pt0 + 8, npt); pt++)
            for (int rb = rb0; rb < std::min(rb0 + 3, nrb); rb++)
              for (int qb = qb0; qb < std::min(qb0 + 6, nqb); qb++)
                if (qb <= 2 * rb + 1) items.push_back(TripleItem{pt * TP_PT, qb * TP_QT, rb * TP_RT, (qb >> 1) == rb ? 1 : 0});
    thc_handle::TripleList l{nPp, NPp, nullptr, (int)items.size()};
    // (+ 4 slots: the gate counter of the launches that use this list lives behind the items)
    if (cudaMalloc(&l.dev, (items.size() + 4) * sizeof(TripleItem)) != cudaSuccess) { check(cudaGetLastError()); return nullptr; }
    // pageable source: the runtime stages the data before returning, so `items` may die at the end of this scope
    check(cudaMemcpyAsync(l.dev, items.data(), items.size() * sizeof(TripleItem), cudaMemcpyHostToDevice, h->stream));
    check(cudaStreamSynchronize(h->stream));
    h->tp_lists.push_back(l);
    return &h->tp_lists.back();
  }
  void triple_product(const double* E, const double* F, const double* G, double* H, i64 nI, i64 nPp, i64 NPp, int accumulate) {
    if (dry || !ok()) return;
    if (!h->smem_configured) {
      check(cudaFuncSetAttribute(triple_product_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, TP_SMEM_BYTES));
      h->smem_configured = true;
    }
    const thc_handle::TripleList* list = triple_items(nPp, NPp);
    CUtensorMap mE, mF, mG;
    if (!list || !make_map3(&mE, E, NPp, nPp, nI) || !make_map3(&mF, F, NPp, nPp, nI) || !make_map3(&mG, G, NPp, NPp, nI)) return;
    TripleParams p;
    p.H = H; p.items = list->dev; p.n_items = list->n;
    p.nI = (int)nI; p.nPp = (int)nPp; p.NPp = (int)NPp; p.accumulate = accumulate;
    const int grid = std::min(list->n, h->sms);
    if (((i64)(list->n + grid - 1) / grid) * nI >= ((i64)1 << 31)) { status = THC_ERR_OVERFLOW; return; }
    // Long launches (>= 64 items per CTA) run gated: a cooperative launch (all CTAs co-resident) in which the CTAs wait
    // for one another every ~16384 grid points of work, so that the L2-ordered work list keeps paying (thc_triple.cuh).
    p.gate = reinterpret_cast<unsigned int*>(list->dev + list->n);
    // Period: 16384 grid points of work, at most 32 items (measured at config 3, step time by period in grid points: none
    // 36.12 s at the power cap, 512 35.29, 2048 34.98, 4096 34.52, 8192 34.27, 16384 34.17: every barrier costs the wait for
    // the slowest CTA, so as rare as keeps the GPU under its power cap).  Short items (nI < 256, config 4) run ungated: a
    // barrier every 16 items of 128 points cost 2.3 % there and the launch is not power-limited.
    p.gate_every = (h->tp_gate && list->n >= 64 * grid && nI >= 256) ? (int)std::max<i64>(1, std::min<i64>(32, 16384 / nI)) : 0;
    prof_start(1, "triple_product", 5.0 * nI * nPp * (double)NPp * NPp);
    if (p.gate_every) {
      check(cudaMemsetAsync(p.gate, 0, sizeof(unsigned int), h->stream));
      void* args[4] = {&mE, &mF, &mG, &p};
      cudaError_t e = cudaLaunchCooperativeKernel(reinterpret_cast<void*>(triple_product_kernel), dim3(grid), dim3(TP_THREADS), args,
                                                  TP_SMEM_BYTES, h->stream);
      if (e != cudaSuccess) {              // not launchable that way here: never gate again on this handle
        cudaGetLastError();
        h->tp_gate = false;
        p.gate_every = 0;
      }
    }
    if (!p.gate_every) triple_product_kernel<<<grid, TP_THREADS, TP_SMEM_BYTES, h->stream>>>(mE, mF, mG, p);
    launched();
    prof_stop(1);
  }
};

}  // namespace thc
