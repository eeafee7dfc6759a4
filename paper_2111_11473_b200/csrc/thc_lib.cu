// C ABI of the THC-RR-CCSD projected doubles residual library (include/thc.h) and the evaluation plan.
//
// The plan is PAPER.md Algorithms 1, 2, 3, 6, 7, 8 (lines 5-10) and 9 re-blocked for one B200:
//   * every contraction over an orbital, Cholesky or grid index is a call of the FP64 DMMA GEMM (thc_gemm.cuh),
//     batched over Cholesky vectors / grid rows so that one launch covers a whole block;
//   * Hadamard products are either fused into a GEMM epilogue (Z .* E^L, Alg.8 line 7 l.792; E .* V, Alg.7
//     lines 14/18 l.757-763) or done by the HBM-streaming kernels of thc_kernels.cuh;
//   * per-P NP x NP Hadamards of Alg.7 line 6 (l.743) and Alg.6 line 1 (l.683) are never materialised: the o x NP
//     factor is row-scaled instead (B^{YZ} = v^{XY} o^{XZ} T^{YZ}  ->  (Xo .* v_X) Z (Xv .* o_X)^T);
//   * Alg.6 line 11 (l.714) runs on the FP64 FMA pipe (triple_product_kernel).
// Notation: P,Q,R amplitude grid (paper W,X,Y,Z), I,J ERI grid, L Cholesky index (paper A); see DESIGN.md.
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include "thc_host.cuh"

using thc::i64;
using thc::Ctx;
using thc::Gemm;

namespace {

struct Inputs {
  const double *Xo, *Xv, *Z, *B_ov, *B_oo;
  const void* B_vv;        // device array, host array or thc_bvv_provider*, per thc_options.bvv_mode (thc.h)
  const double *Y, *V, *eps;
  const double* t1 = nullptr;    // [o][v] singles amplitudes: T1-dressed evaluation, else NULL
};
struct Outputs {
  double* R;
  double* terms[6];   // s1 s2 s3 s6 s7 s9 (NULL -> scratch)
  double* xi_oo;
  double* xi_vv;
  double* sigma = nullptr;                         // [o][v] singles residual (T1 evaluation only)
  double* sigma_parts[2] = {nullptr, nullptr};     // Omega G+H (Eq.38), Omega I+J (Eq.42)
};
// Sharded evaluation: phase 1 computes one rank's partial
// sums over its Cholesky range [Lb, Le) and its rows [Pb, Pe) of the T2^2 terms into `packed`; after the caller has
// summed `packed` over the ranks, phase 2 finishes (Alg.3 tail, Alg.9, the C7 V C7^T part of Alg.7, the sum).
// phase 0 is the ordinary single-device evaluation.  Packed layout: thc_shard_doubles().
struct Shard {
  int phase = 0;
  i64 Lb = 0, Le = 0, Pb = 0, Pe = 0;
  double* packed = nullptr;
};
struct PackedLayout {
  i64 s1, s2, C3, s6, s7, C7, xi_oo, xi_vv, total;
  PackedLayout(i64 o, i64 v, i64 NP, i64 NX) {
    const i64 NP2 = NP * NP;
    s1 = 0; s2 = NP2; C3 = 2 * NP2; s6 = 3 * NP2; s7 = 4 * NP2; C7 = 5 * NP2; xi_oo = C7 + NP * NX; xi_vv = xi_oo + o * o;
    total = xi_vv + v * v;
  }
};

inline i64 pad_to(i64 x, i64 m) { return (x + m - 1) / m * m; }

// O(N^5) GEMM-only evaluation of the ladder-type T2^2 terms: PAPER.md Alg.4 (Eq.32, l.608-643) and Alg.5 (Eq.33,
// l.645-680), the variant the paper prefers for small molecules (l.250, l.309).  Every line of the listings is a GEMM
// batched over a block of pairs -- (i, j) for Alg.4, (a, j) for Alg.5 -- with the Hadamard products of lines 4, 7, 10 fused
// into GEMM epilogues (aux) and line 13 done by pair_accumulate_kernel.  Lines 3-5 of both algorithms are the explicit
// amplitudes of the pair, t_ij^cd and t_lj^ad, formed from the scaled factors XS[(i,a)][P] = Xo[i,P] Xv[a,P].
void plan_s6_n5(Ctx& c, const Inputs& in, double* s6, const double* XoT, const double* XvT, const double* YoT, const double* YvT) {
  thc_handle* h = c.h;
  thc::Arena& ar = c.ar;
  const i64 o = h->o, v = h->v, NP = h->NP, NX = h->NX, NP2 = NP * NP, ov = o * v;
  const double* Yo = in.Y;
  const double* Yv = in.Y + o * NX;
  const double *Z = in.Z, *V = in.V, *Xo = in.Xo, *Xv = in.Xv;
  const i64 m0 = ar.mark();
  c.fill(s6, NP2, 0.0);
  double* XS = ar.alloc(ov * NP);
  c.rowscale(Xv, NP, Xo, NP, nullptr, 1.0, XS, o, v, NP);                       // XS[(i,a)][P]
  double *E = ar.alloc(o * NX * NX), *W = ar.alloc(o * o * NX);                // one i (or a) at a time: lines 6-8
  const i64 budget = (i64)3 << 30;                                              // bytes of per-block intermediates
  // ---- Alg.4: pairs (i, j), blocks of ni values of i -------------------------------------------------------------------------
  {
    const i64 per = 8 * (v * NP + v * ov + v * o * NX + o * o * o + o * o * NP + o * NP2 + ov * NP + ov * v);
    const i64 bi = std::max<i64>(1, std::min<i64>(o, budget / per));
    for (i64 i0 = 0; i0 < o; i0 += bi) {
      const i64 ni = std::min<i64>(bi, o - i0), m1 = ar.mark();
      double *A3b = ar.alloc(ni * v * NP), *T4 = ar.alloc(ni * v * ov), *U1 = ar.alloc(ni * v * o * NX), *X4 = ar.alloc(ni * o * o * o);
      c.gemm(Gemm(XS + i0 * v * NP, NP, 'K', Z, NP, 'K', A3b, NP, ni * v, NP, NP));             // lines 3-4: T .* A folded into XS Z
      c.gemm(Gemm(A3b, NP, 'K', XS, NP, 'K', T4, ov, ni * v, ov, NP));                         // line 5: T4[(i,c)][(j,d)] = t_ij^cd
      c.gemm(Gemm(T4, v, 'K', YvT, v, 'K', U1, NX, ni * v * o, NX, v));                        // line 6, first half: sum_d
      for (i64 ii = 0; ii < ni; ii++) {
        // line 6 (second half) + line 7: E^{IJ} = z^{IJ} sum_c x_c^I U1[(i,c,j)][J], batch over j
        c.gemm(Gemm(YvT, v, 'K', U1 + ii * v * o * NX, o * NX, 'N', E, NX, NX, NX, v).batch(o, 0, NX, NX * NX).aux(V, NX, 0));
        // line 8: F_kl = sum_IJ E^{IJ} x_k^I x_l^J
        c.gemm(Gemm(Yo, NX, 'K', E, NX, 'N', W, NX, o, NX, NX).batch(o, 0, NX * NX, o * NX));
        c.gemm(Gemm(W, NX, 'K', Yo, NX, 'K', X4 + ii * o * o * o, o, o * o, o, NX));
      }
      double *FX = ar.alloc(ni * o * o * NP), *Hb = ar.alloc(ni * o * NP2), *HX = ar.alloc(ni * ov * NP), *I4 = ar.alloc(ni * ov * v);
      c.gemm(Gemm(X4, o, 'K', XoT, o, 'K', FX, NP, ni * o * o, NP, o));                        // line 9, first half: sum_l
      c.gemm(Gemm(Xo, NP, 'M', FX, NP, 'N', Hb, NP, NP, NP, o).batch(ni * o, 0, o * NP, NP2).aux(Z, NP, 0));   // lines 9-10: H = T .* G
      c.gemm(Gemm(Xv, NP, 'K', Hb, NP, 'N', HX, NP, v, NP, NP).batch(ni * o, 0, NP2, v * NP));                  // line 11: sum_Y
      c.gemm(Gemm(HX, NP, 'K', Xv, NP, 'K', I4, v, ni * ov, v, NP));                                          //          sum_Y' -> I_ab
      c.gemm(Gemm(I4, v, 'K', XvT, v, 'K', HX, NP, ni * ov, NP, v));                                          // line 12: sum_b
      c.gemm(Gemm(Xv, NP, 'M', HX, NP, 'N', Hb, NP, NP, NP, v).batch(ni * o, 0, v * NP, NP2));                  //          sum_a -> J^{XX'}
      c.pair_accumulate(Hb, Xo + i0 * NP, NP, Xo, NP, s6, NP, ni, o);                                          // line 13
      ar.release(m1);
    }
  }
  // ---- Alg.5: pairs (a, j), blocks of na values of a -------------------------------------------------------------------------
  {
    const i64 per = 8 * (2 * o * NP + o * ov + o * o * NX + o * ov + 2 * o * o * NP + o * NP2 + o * ov);
    const i64 ba = std::max<i64>(1, std::min<i64>(v, budget / per));
    for (i64 a0 = 0; a0 < v; a0 += ba) {
      const i64 na = std::min<i64>(ba, v - a0), m1 = ar.mark();
      double *XSa = ar.alloc(na * o * NP), *A3a = ar.alloc(na * o * NP), *T4a = ar.alloc(na * o * ov), *U5 = ar.alloc(na * o * o * NX);
      double* F5 = ar.alloc(na * o * ov);
      c.rowscale(Xo, NP, Xv + a0 * NP, NP, nullptr, 1.0, XSa, na, o, NP);                       // XSa[(a,l)][P]
      c.gemm(Gemm(XSa, NP, 'K', Z, NP, 'K', A3a, NP, na * o, NP, NP));
      c.gemm(Gemm(A3a, NP, 'K', XS, NP, 'K', T4a, ov, na * o, ov, NP));                        // lines 3-5: T4a[(a,l)][(j,d)] = t_lj^ad
      c.gemm(Gemm(T4a, v, 'K', YvT, v, 'K', U5, NX, na * o * o, NX, v));                       // line 6, first half: sum_d
      for (i64 aa = 0; aa < na; aa++) {
        c.gemm(Gemm(YoT, o, 'K', U5 + aa * o * o * NX, o * NX, 'N', E, NX, NX, NX, o).batch(o, 0, NX, NX * NX).aux(V, NX, 0));   // lines 6-7
        c.gemm(Gemm(Yo, NX, 'K', E, NX, 'K', W, NX, o, NX, NX).batch(o, 0, NX * NX, o * NX));                               // line 8: sum_J x_k^J
        c.gemm(Gemm(W, NX, 'K', Yv, NX, 'K', F5 + aa * o * ov, v, o * o, v, NX));                                          //         sum_I x_c^I
      }
      double *FY = ar.alloc(na * o * o * NP), *Hb = ar.alloc(na * o * NP2), *HX = ar.alloc(na * o * o * NP), *I5 = ar.alloc(na * o * ov);
      c.gemm(Gemm(F5, v, 'K', XvT, v, 'K', FY, NP, na * o * o, NP, v));                        // line 9, first half: sum_c
      c.gemm(Gemm(FY, NP, 'M', Xo, NP, 'N', Hb, NP, NP, NP, o).batch(na * o, o * NP, 0, NP2).aux(Z, NP, 0));   // lines 9-10
      c.gemm(Gemm(Xo, NP, 'K', Hb, NP, 'N', HX, NP, o, NP, NP).batch(na * o, 0, NP2, o * NP));                  // line 11: sum_Y y_i^Y
      c.gemm(Gemm(HX, NP, 'K', Xv, NP, 'K', I5, v, na * o * o, v, NP));                                        //          sum_Y' y_b^Y' -> I_ib
      c.gemm(Gemm(I5, v, 'K', XvT, v, 'K', HX, NP, na * o * o, NP, v));                                        // line 12: sum_b
      c.gemm(Gemm(Xo, NP, 'M', HX, NP, 'N', Hb, NP, NP, NP, o).batch(na * o, 0, o * NP, NP2));                  //          sum_i -> J^{XX'}
      c.pair_accumulate(Hb, Xv + a0 * NP, NP, Xo, NP, s6, NP, na, o);                                          // line 13: A = y_a^X y_j^X'
      ar.release(m1);
    }
  }
  ar.release(m0);
}

// The whole residual evaluation.  Runs either for real or dry (workspace sizing); both take identical branches.
void plan_residual(Ctx& c, const Inputs& in, const Outputs& out, const Shard& sh = Shard()) {
  thc_handle* h = c.h;
  thc::Arena& ar = c.ar;
  const i64 o = h->o, v = h->v, NP = h->NP, NX = h->NX;
  const bool local = sh.phase != 2;        // the L loop and the row blocks of Alg.6 / Alg.7
  const bool post = sh.phase != 1;         // everything that needs the rank-summed intermediates
  const i64 Lb = sh.phase ? sh.Lb : 0, Le = sh.phase ? sh.Le : h->NL, NL = Le - Lb;     // B_* point at vector Lb
  const i64 Pb = sh.phase ? sh.Pb : 0, Pe = sh.phase ? sh.Pe : NP;
  const PackedLayout pk(o, v, NP, NX);
  const i64 NP2 = NP * NP, ov = o * v;
  const int mask = h->term_mask ? h->term_mask : THC_TERM_ALL;
  const bool do_s1 = mask & THC_TERM_S1, do_s2 = mask & THC_TERM_S2, do_s3 = mask & THC_TERM_S3;
  const bool do_s6 = mask & THC_TERM_S6, do_s7 = mask & THC_TERM_S7, do_s9 = mask & THC_TERM_S9;
  const double* Yo = in.Y;
  const double* Yv = in.Y + o * NX;

  // ---- persistent buffers -----------------------------------------------------------------------------------------
  double* term[6];
  for (int k = 0; k < 6; k++) term[k] = out.terms[k] ? out.terms[k] : (sh.phase == 1 && (k == 2 || k == 5) ? nullptr : ar.alloc(NP2));
  double* xi_oo = out.xi_oo ? out.xi_oo : ar.alloc(o * o);
  double* xi_vv = out.xi_vv ? out.xi_vv : ar.alloc(v * v);
  if (sh.phase) {                          // the summed quantities live in the packed buffer
    term[0] = sh.packed + pk.s1; term[1] = sh.packed + pk.s2; term[3] = sh.packed + pk.s6; term[4] = sh.packed + pk.s7;
    xi_oo = sh.packed + pk.xi_oo; xi_vv = sh.packed + pk.xi_vv;
  }
  double *s1 = term[0], *s2 = term[1], *s3 = term[2], *s6 = term[3], *s7 = term[4], *s9 = term[5];
  double* XoT = ar.alloc(NP * o);
  double* XvT = ar.alloc(NP * v);
  double* YoT = ar.alloc(NX * o);
  double* YvT = ar.alloc(NX * v);
  double *omat = ar.alloc(NP2), *vmat = ar.alloc(NP2), *wmat = ar.alloc(NP2), *Kmat = ar.alloc(NP2);
  double* C3 = sh.phase ? sh.packed + pk.C3 : ar.alloc(NP2);
  double *Aa = ar.alloc(std::max<i64>(NL, 1) * NP), *Dm = ar.alloc(std::max<i64>(NL, 1) * NP);

  // T1-dressed evaluation (phase 0 only): accumulators of the dressed Fock matrix minus diag(eps), in the layouts the
  // later steps read (Fd_oo[i][j] = F^_ij, FdT_vv[b][a] = F^_ab, F_ov[i][a], F_voT[i][a] = F^_ai), and of the singles
  // residual.  F^_pq = (Xp^T diag(eps) Xh)_pq + sum_L [ 2 B^_pq tau^L - sum_kc (pc|kq)^-like exchange ], tau^L = sum_kc B_kc t_k^c.
  const double* t1 = sh.phase == 0 ? in.t1 : nullptr;
  double *Fd_oo = nullptr, *FdT_vv = nullptr, *F_ov = nullptr, *F_voT = nullptr, *sigGH = nullptr, *sigIJ = nullptr, *Abar = nullptr;
  if (t1) {
    Fd_oo = ar.alloc(o * o); FdT_vv = ar.alloc(v * v); F_ov = ar.alloc(ov); F_voT = ar.alloc(ov);
    sigGH = out.sigma_parts[0] ? out.sigma_parts[0] : ar.alloc(ov);
    sigIJ = out.sigma_parts[1] ? out.sigma_parts[1] : ar.alloc(ov);
    Abar = ar.alloc(std::max<i64>(NL, 1) * NP);
  }

  // ---- H0: transposed factors and grams (Alg.1 l.481-485) ------------------------------------------------------------
  c.transpose(in.Xo, XoT, o, NP);
  c.transpose(in.Xv, XvT, v, NP);
  c.transpose(Yo, YoT, o, NX);
  c.transpose(Yv, YvT, v, NX);
  c.gemm(Gemm(XoT, o, 'K', XoT, o, 'K', omat, NP, NP, NP, o));
  c.gemm(Gemm(XvT, v, 'K', XvT, v, 'K', vmat, NP, NP, NP, v));
  c.hadamard(omat, vmat, wmat, NP2);                                         // w = o .* v
  c.gemm(Gemm(wmat, NP, 'K', in.Z, NP, 'K', Kmat, NP, NP, NP, NP));           // K = w Z   (Z symmetric)
  if (local) {
    if (sh.phase == 1) c.fill(sh.packed, pk.total, 0.0);      // rows / terms this rank does not own stay zero
    c.fill(C3, NP2, 0.0);
    c.fill(s1, NP2, 0.0);
    c.fill(xi_oo, o * o, 0.0);
    c.fill(xi_vv, v * v, 0.0);
    if (t1) {
      c.fill(Fd_oo, o * o, 0.0); c.fill(FdT_vv, v * v, 0.0); c.fill(F_ov, ov, 0.0); c.fill(sigGH, ov, 0.0);
      c.t1_eps(in.eps, t1, F_voT, o, v);                 // (eps_a - eps_i) t_i^a: Xp^T diag(eps) Xh, vo block
    }
  }

  // ---- L-block loop: Alg.1 + Alg.3 (H1-H4) and Alg.2 + Alg.8 (H5-H6) fused over the Cholesky index (l.238) ---------
  const bool need_ladder = local && (do_s1 || do_s3);
  const bool need_ring = local && (do_s2 || do_s9 || t1);
  const bool need_bvv = need_ladder || t1;       // the dressed vv blocks also feed the singles residual and F^
  // B_vv source: resident (device pointer), or streamed one L-block at a time into a double buffer (l.191-195)
  const bool streamed = h->bvv_mode != THC_BVV_DEVICE && need_bvv;
  double* bvv_buf[2] = {nullptr, nullptr};
  if (streamed) { bvv_buf[0] = ar.alloc(h->bL * v * v); bvv_buf[1] = ar.alloc(h->bL * v * v); }
  if (streamed && !c.dry) c.bvv_begin();
  if (streamed && !c.dry && h->bvv_mode == THC_BVV_HOST)
    c.bvv_copy(bvv_buf[0], static_cast<const double*>(in.B_vv), 0, std::min<i64>(h->bL, NL), v, 0);
  i64 blk = 0;
  for (i64 L0 = 0; L0 < NL; L0 += h->bL, blk++) {
    const i64 nl = std::min<i64>(h->bL, NL - L0);
    const i64 mT = ar.mark();
    const double* bvv = static_cast<const double*>(in.B_vv) + L0 * v * v;
    if (streamed) {
      bvv = bvv_buf[blk & 1];
      if (!c.dry) {
        if (h->bvv_mode == THC_BVV_HOST) {
          const i64 L1 = L0 + h->bL;                 // prefetch the next block while this one is consumed
          if (L1 < NL) c.bvv_copy(bvv_buf[(blk + 1) & 1], static_cast<const double*>(in.B_vv), L1, std::min<i64>(h->bL, NL - L1), v, blk + 1);
          c.bvv_wait_loaded(blk);
        } else {
          c.bvv_provide(static_cast<const thc_bvv_provider*>(in.B_vv), Lb + L0, nl, bvv_buf[blk & 1]);
        }
      }
    }
    // ---- T1 dressing of this block (Eqs.25-27 l.203-209 in the MO basis).  Index order matters now (l.211).  Projecting
    // Eq.28 term by term gives C^L = v .* Bbar^T - o .* Btilde with Bbar^{XY} = sum_ki y_k^X l_ki y_i^Y and
    // Btilde^{XY} = sum_ac y_a^X l_ac y_c^Y (at t1 = 0 the transpose is invisible; Alg.1 lines 6-8 as printed pair X with
    // the first index of l_ki, which the determinant-space pin of oracle/t1.py rules out), and Eq.38 gives
    // -sum_k l_ki D_ka for Alg.8 line 12.  The half-transforms below contract the SECOND index of a stored block first,
    // so the dressed oo block is kept in natural order (Boo_h[l][k][j] = B^_kj -> Mo = Bbar^T) and the dressed vv block
    // transposed (BvvT[l][c][a] = B^_ac -> Mv = Btilde).
    const double* boo = in.B_oo + L0 * o * o;
    const double* bov = in.B_ov + L0 * ov;
    double *TL = nullptr, *Boo_h = nullptr, *BvvT = nullptr, *BvoT = nullptr, *Sl = nullptr, *tau = nullptr;
    if (t1) {
      TL = ar.alloc(nl * o * o); Boo_h = ar.alloc(nl * o * o); BvoT = ar.alloc(nl * ov); Sl = ar.alloc(nl * v * o); tau = ar.alloc(nl);
      BvvT = streamed ? bvv_buf[blk & 1] : ar.alloc(nl * v * v);       // a streamed block is ours: dress it in place
      // TL[l][k][j] = sum_a B_ka t_j^a ;  B^_kj = B_kj + TL[l][k][j]
      c.gemm(Gemm(bov, v, 'K', t1, v, 'K', TL, o, nl * o, o, v));
      c.axpby(boo, TL, 1.0, 1.0, Boo_h, nl * o * o);
      // B^_ac = B_ac - sum_i t_i^a B_ic, stored as BvvT[l][c][a]
      if (!streamed) c.copy(bvv, BvvT, nl * v * v);
      c.gemm(Gemm(bov, v, 'M', t1, v, 'N', BvvT, v, v, v, o).batch(nl, ov, 0, v * v).ab(-1.0, 1.0));
      // tau^l = sum_kc B_kc t_k^c ;  Sl[l][a][k] = sum_c B^_ac t_k^c
      c.rowdot(t1, ov, bov, ov, ov, tau, 1, nl, 1, ov);
      c.gemm(Gemm(BvvT, v, 'M', t1, v, 'K', Sl, o, v, o, v).batch(nl, v * v, 0, v * o));
      // B^_ai = B_ia - sum_j t_j^a B_ji + sum_b B^_ab t_i^b, stored as BvoT[l][i][a]
      c.copy(bov, BvoT, nl * ov);
      c.gemm(Gemm(boo, o, 'K', t1, v, 'N', BvoT, v, o, v, o).batch(nl, o * o, 0, ov).ab(-1.0, 1.0));
      c.gemm(Gemm(t1, v, 'K', BvvT, v, 'N', BvoT, v, o, v, v).batch(nl, 0, v * v, ov).ab(1.0, 1.0));
      // dressed Fock matrix: 2 tau^l B^ parts (one GEMV-shaped product over l each) and the exchange parts
      c.gemm(Gemm(tau, nl, 'K', Boo_h, o * o, 'N', Fd_oo, o * o, 1, o * o, nl).ab(2.0, 1.0));
      c.gemm(Gemm(TL, o, 'K', Boo_h, o, 'N', Fd_oo, o, o, o, o).kbatch(nl, o * o, o * o).ab(-1.0, 1.0));       // sum_k T[i][k] B^_kj
      c.gemm(Gemm(tau, nl, 'K', BvvT, v * v, 'N', FdT_vv, v * v, 1, v * v, nl).ab(2.0, 1.0));
      c.gemm(Gemm(bov, v, 'M', Sl, o, 'K', FdT_vv, v, v, v, o).kbatch(nl, ov, v * o).ab(-1.0, 1.0));         // sum_k B_kb S[a][k]
      c.gemm(Gemm(tau, nl, 'K', bov, ov, 'N', F_ov, ov, 1, ov, nl).ab(2.0, 1.0));
      c.gemm(Gemm(TL, o, 'K', bov, v, 'N', F_ov, v, o, v, o).kbatch(nl, o * o, ov).ab(-1.0, 1.0));            // sum_k T[i][k] B_ka
      c.gemm(Gemm(tau, nl, 'K', BvoT, ov, 'N', F_voT, ov, 1, ov, nl).ab(2.0, 1.0));
      c.gemm(Gemm(Boo_h, o, 'M', Sl, o, 'K', F_voT, v, o, v, o).kbatch(nl, o * o, v * o).ab(-1.0, 1.0));      // sum_k B^_ki S[a][k]
      boo = Boo_h;
      bvv = BvvT;
    }
    const i64 m0 = ar.mark();
    if (need_ladder) {
      double* T1T = ar.alloc(NP * nl * o);
      double* T2T = ar.alloc(NP * nl * v);
      double *Mo = ar.alloc(nl * NP2), *Mv = ar.alloc(nl * NP2);
      // H1: T1T[P][(l,j)] = sum_i Xo[i,P] B^l_ij ;  Mo^l[P][Q] = sum_j T1T[P][(l,j)] Xo[j,Q]      (Alg.1 lines 6-7)
      c.gemm(Gemm(XoT, o, 'K', boo, o, 'K', T1T, nl * o, NP, nl * o, o));
      // (B^l symmetric => M^{o,l}, M^{v,l} symmetric: for NP of several tiles only the upper tiles are computed and the
      //  lower ones mirrored in one batched pass; for small NP the mirror pass costs more than it saves)
      const bool sym_half = NP >= 640 && !t1;          // dressed vectors are not symmetric (l.211)
      Gemm gMo = Gemm(T1T, nl * o, 'K', XoT, o, 'K', Mo, NP, NP, NP, o).batch(nl, o, 0, NP2);
      c.gemm(sym_half ? gMo.upper_only() : gMo);
      // H2: same with the vv block                                                                  (Alg.1 lines 10-11)
      c.gemm(Gemm(XvT, v, 'K', bvv, v, 'K', T2T, nl * v, NP, nl * v, v));
      if (streamed && !c.dry && h->bvv_mode == THC_BVV_HOST && !t1) c.bvv_release(blk);
      Gemm gMv = Gemm(T2T, nl * v, 'K', XvT, v, 'K', Mv, NP, NP, NP, v).batch(nl, v, 0, NP2);
      c.gemm(sym_half ? gMv.upper_only() : gMv);
      if (sym_half) { c.mirror_upper(Mo, NP, nl); c.mirror_upper(Mv, NP, nl); }
      // H3: C^l = v .* Mo^l - o .* Mv^l (in place over Mo);  C3 += Mo^l .* Mv^l                   (Alg.1 l.8,12,13; Alg.3 l.7)
      c.combine(Mo, Mv, omat, vmat, C3, NP2, nl);
      if (do_s1) {
        // H4: D^l = C^l Z ;  s1 += sum_l D^l C^l^T                                                   (Alg.1 lines 14-15)
        double* D = Mv;   // Mv is dead after the combine
        c.gemm(Gemm(Mo, NP, 'K', in.Z, NP, 'K', D, NP, nl * NP, NP, NP));
        // (sigma1 = sum_l C^l Z C^l^T is symmetric: only the tiles on and above the diagonal are computed)
        c.gemm(Gemm(D, NP, 'K', Mo, NP, 'K', s1, NP, NP, NP, NP).kbatch(nl, NP2, NP2).ab(1.0, 1.0).upper_only());
      }
      ar.release(m0);
    }
    if (need_ring) {
      // H5: TT[Q][(l,i)] = sum_a Xv[a,Q] B^l_ia ;  a^l_P = sum_i Xo[i,P] TT[P][(l,i)]              (Alg.8 line 5 l.788)
      double* TT = ar.alloc(NP * nl * o);
      c.gemm(Gemm(XvT, v, 'K', in.B_ov + L0 * ov, v, 'K', TT, nl * o, NP, nl * o, v));
      c.rowdot(XoT, o, TT, o, nl * o, Aa + L0 * NP, NP, nl, NP, o);
      // W^l = Z .* E^l,  E^l[P][Q] = sum_i Xo[i,P] TT[Q][(l,i)]                                     (Alg.8 lines 6-7)
      double* W = ar.alloc(nl * NP2);
      c.gemm(Gemm(XoT, o, 'K', TT, nl * o, 'K', W, NP, NP, NP, o).batch(nl, 0, o, NP2).aux(in.Z, NP, 0));
      double* ZA = ar.alloc(nl * NP);
      c.gemm(Gemm(Aa + L0 * NP, NP, 'K', in.Z, NP, 'K', ZA, NP, nl, NP, NP));
      // H6: D^l_ia = sum_PQ Xo[i,Q] Xv[a,P] N^l_PQ,  N^l = 2 diag(Z a^l) - W^l                      (Alg.8 line 8 l.794)
      double* G1 = ar.alloc(o * nl * NP);
      c.gemm(Gemm(in.Xo, NP, 'K', W, NP, 'K', G1, nl * NP, o, nl * NP, NP));
      c.qm(G1, in.Xo, ZA, o, nl, NP);
      double* Dia = ar.alloc(nl * ov);
      c.gemm(Gemm(G1, nl * NP, 'K', in.Xv, NP, 'K', Dia, v, o, v, NP).batch(nl, NP, 0, ov));
      // xi_ij += sum_a B^l_ia D^l_ja ;  xi_ab -= sum_i D^l_ia B^l_ib                               (Alg.8 lines 9-10; Eqs.39-40)
      c.gemm(Gemm(in.B_ov + L0 * ov, v, 'K', Dia, v, 'K', xi_oo, o, o, o, v).kbatch(nl, ov, ov).ab(1.0, 1.0));
      c.gemm(Gemm(Dia, v, 'M', in.B_ov + L0 * ov, v, 'N', xi_vv, v, v, v, nl * o).ab(-1.0, 1.0));
      // d^l_P = sum_ia Xo[i,P] Xv[a,P] D^l_ia                                                         (Alg.2 lines 8, 12)
      double* DX = ar.alloc(nl * o * NP);
      c.gemm(Gemm(Dia, v, 'K', XvT, v, 'K', DX, NP, nl * o, NP, v));
      c.coldot(in.Xo, NP, DX, o * NP, NP, Dm + L0 * NP, NP, nl, NP, o);
      if (t1) {
        // A-bar^l_P = sum_ia Xo[i,P] Xv[a,P] B^_ai                                                       (Eq.30 l.229; Alg.2 line 4)
        c.gemm(Gemm(XvT, v, 'K', BvoT, v, 'K', TT, nl * o, NP, nl * o, v));
        c.rowdot(XoT, o, TT, o, nl * o, Abar + L0 * NP, NP, nl, NP, o);
        // Omega G, H: sigma_ia += sum_b D^l_ib B^_ab - sum_k B^_ki D^l_ka                                (Alg.8 lines 11-12 l.800-803; Eq.38)
        c.gemm(Gemm(Dia, v, 'K', BvvT, v, 'N', sigGH, v, o, v, v).kbatch(nl, ov, v * v).ab(1.0, 1.0));
        c.gemm(Gemm(Boo_h, o, 'M', Dia, v, 'N', sigGH, v, o, v, o).kbatch(nl, o * o, ov).ab(-1.0, 1.0));         // sum_k B^_ki D_ka
      }
      ar.release(m0);
    }
    if (streamed && !c.dry && h->bvv_mode == THC_BVV_HOST && t1) c.bvv_release(blk);     // the dressed block was read until here
    ar.release(mT);
  }

  if (local && do_s1) c.mirror_upper(s1, NP);          // complete the symmetric sigma1 from its upper triangle

  // ---- H7: s2 = A A^T + Dm A^T + A Dm^T  (Alg.2 line 13 l.559; rows of Aa/Dm are Cholesky vectors) --------------------
  if (!local) {
    // phase 2: s2 arrives summed over the ranks
  } else if (do_s2 && NL > 0) {
    const i64 m0 = ar.mark();
    // (T1: the bare term and the partners of D use A-bar from the dressed vo block, Alg.2 line 14 l.559; Dm comes from l_ia)
    const double* A2 = t1 ? Abar : Aa;
    double* AD = ar.alloc(NL * NP);
    c.axpby(A2, Dm, 1.0, 1.0, AD, NL * NP);
    c.gemm(Gemm(AD, NP, 'M', A2, NP, 'N', s2, NP, NP, NP, NL));
    c.gemm(Gemm(A2, NP, 'M', Dm, NP, 'N', s2, NP, NP, NP, NL).ab(1.0, 1.0));
    ar.release(m0);
  } else {
    c.fill(s2, NP2, 0.0);
  }

  // ---- H8: Alg.3 tail and Alg.9 ------------------------------------------------------------------------------------
  if (!post) {
    // phase 1: Alg.3 tail and Alg.9 need the rank-summed C3, xi_oo, xi_vv
  } else if (do_s3) {
    // s3 = -(K C3^T + C3 K^T)                                                                        (Alg.3 line 12 l.601)
    const i64 m0 = ar.mark();
    double* P3 = ar.alloc(NP2);
    c.gemm(Gemm(Kmat, NP, 'K', C3, NP, 'K', P3, NP, NP, NP, NP));
    c.symmetrize(P3, s3, NP, -1.0);
    ar.release(m0);
  } else {
    c.fill(s3, NP2, 0.0);
  }
  if (!post) {
  } else if (do_s9) {
    // F'_oo = diag(eps_o) + xi_oo, F'_vv = diag(eps_v) + xi_vv; o~ = Xo^T F'_oo^T.. (Alg.9 lines 5-10 l.823-839)
    const i64 m0 = ar.mark();
    double *FooT = ar.alloc(o * o), *Fvv = ar.alloc(v * v);
    double *CoT = ar.alloc(NP * o), *DvT = ar.alloc(NP * v), *otil = ar.alloc(NP2), *vtil = ar.alloc(NP2);
    double *E9 = ar.alloc(NP2), *P9 = ar.alloc(NP2);
    if (t1) {                                   // F' = F^ + xi: add the dressing parts to copies of xi before the diagonal
      double *Xoo = ar.alloc(o * o), *Xvv = ar.alloc(v * v);
      c.axpby(xi_oo, Fd_oo, 1.0, 1.0, Xoo, o * o);
      c.transpose(FdT_vv, Xvv, v, v);
      c.axpby(Xvv, xi_vv, 1.0, 1.0, Xvv, v * v);
      c.fock(in.eps, Xoo, Xvv, FooT, Fvv, o, v);
    } else {
      c.fock(in.eps, xi_oo, xi_vv, FooT, Fvv, o, v);
    }
    c.gemm(Gemm(XoT, o, 'K', FooT, o, 'K', CoT, o, NP, o, o));         // CoT[P][i] = sum_j Xo[j,P] F'[j][i]
    c.gemm(Gemm(XoT, o, 'K', CoT, o, 'K', otil, NP, NP, NP, o));       // o~[P][Q] = sum_i Xo[i,P] C_i^Q
    c.gemm(Gemm(XvT, v, 'K', Fvv, v, 'K', DvT, v, NP, v, v));          // DvT[P][a] = sum_b Xv[b,P] F'[a][b]
    c.gemm(Gemm(XvT, v, 'K', DvT, v, 'K', vtil, NP, NP, NP, v));
    c.had2_diff(omat, vtil, otil, vmat, E9, NP2);                       // E = o .* v~ - o~ .* v
    c.gemm(Gemm(E9, NP, 'K', Kmat, NP, 'K', P9, NP, NP, NP, NP));       // E K^T
    c.symmetrize(P9, s9, NP, 1.0);
    ar.release(m0);
  } else {
    c.fill(s9, NP2, 0.0);
  }

  // ---- H10: Alg.7, ring-type T2^2 terms with THC ERIs (Eqs.35-37 l.261-271; prefactor 1/2, R2) -----------
  if (do_s7) {
    const i64 m0 = ar.mark();
    double* C7 = sh.phase ? sh.packed + pk.C7 : ar.alloc(NP * NX);
    double *Rb = nullptr, *Sb = nullptr;
    if (local) { Rb = ar.alloc(NP * ov); Sb = ar.alloc(NP * ov); }
    // pass 1 (Alg.7 lines 3-7): S^P = -(Xo .* v_P) Z (Xv .* o_P)^T ;  R^P = 2 (Xo .* K_P) Xv^T + S^P
    const i64 bA = std::min<i64>(NP, h->bP7 * 16);
    for (i64 P0 = 0; local && P0 < NP; P0 += bA) {          // R^Q, S^Q are needed for every Q on every rank
      const i64 npb = std::min<i64>(bA, NP - P0), m1 = ar.mark();
      double *XoV = ar.alloc(npb * o * NP), *SZ = ar.alloc(npb * o * NP);
      c.rowscale(in.Xo, NP, vmat + P0 * NP, NP, nullptr, 1.0, XoV, npb, o, NP);
      c.gemm(Gemm(XoV, NP, 'K', in.Z, NP, 'K', SZ, NP, npb * o, NP, NP));
      c.rowscale_inplace(SZ, omat + P0 * NP, NP, -1.0, npb, o, NP);
      c.gemm(Gemm(SZ, NP, 'K', in.Xv, NP, 'K', Sb + P0 * ov, v, npb * o, v, NP));
      c.rowscale(in.Xo, NP, Kmat + P0 * NP, NP, SZ, 2.0, XoV, npb, o, NP);         // RA (reuses XoV)
      c.gemm(Gemm(XoV, NP, 'K', in.Xv, NP, 'K', Rb + P0 * ov, v, npb * o, v, NP));
      ar.release(m1);
    }
    // pass 2 (lines 9-19): per P, E = Yo^T R^P Yv, F = E .* V, G^P = Yo F^T Yv^T; rows of s7 from G R^T and G~ S^T
    for (i64 P0 = Pb; local && P0 < Pe; P0 += h->bP7) {      // this rank's rows of sigma7
      const i64 npb = std::min<i64>(h->bP7, Pe - P0), m1 = ar.mark();
      const bool fused = Ctx::ring_supported(o);       // E and F = E .* V stay in registers (thc_ring.cuh)
      double *RYT = ar.alloc(npb * NX * o), *EF = fused ? nullptr : ar.alloc(npb * NX * NX), *FYT = ar.alloc(npb * o * NX), *Gb = ar.alloc(npb * ov);
      for (int pass = 0; pass < 2; pass++) {
        const double* src = pass == 0 ? Rb : Sb;
        c.gemm(Gemm(YvT, v, 'K', src + P0 * ov, v, 'K', RYT, o, NX, o, v).batch(npb, 0, ov, NX * o));
        if (pass == 0) c.rowdot(YoT, o, RYT, NX * o, o, C7 + P0 * NX, NX, npb, NX, o);     // line 9
        if (fused) {
          c.ring_fused(YoT, RYT, in.V, Yo, FYT, NX, o, npb);
        } else {
          c.gemm(Gemm(YoT, o, 'K', RYT, o, 'K', EF, NX, NX, NX, o).batch(npb, 0, NX * o, NX * NX).aux(in.V, NX, 0));
          c.gemm(Gemm(Yo, NX, 'K', EF, NX, 'K', FYT, NX, o, NX, NX).batch(npb, 0, NX * NX, o * NX));
        }
        c.gemm(Gemm(FYT, NX, 'K', Yv, NX, 'K', Gb, v, npb * o, v, NX));
        c.gemm(Gemm(Gb, ov, 'K', src, ov, 'K', s7 + P0 * NP, NP, npb, NP, ov).ab(pass == 0 ? -0.5 : 0.5, pass == 0 ? 0.0 : 1.0));
      }
      ar.release(m1);
    }
    // line 10 + first part of line 22: s7 += C7 V C7^T  (needs every row of C7: after the rank sum)
    if (post) {
      double* CV = ar.alloc(NP * NX);
      c.gemm(Gemm(C7, NX, 'K', in.V, NX, 'K', CV, NX, NP, NX, NX));
      c.gemm(Gemm(CV, NX, 'K', C7, NX, 'K', s7, NP, NP, NP, NX).ab(1.0, 1.0));
    }
    ar.release(m0);
  } else if (sh.phase == 0) {
    c.fill(s7, NP2, 0.0);
  }

  // ---- H9: Alg.6, ladder-type T2^2 terms with THC ERIs (Eq.34 l.254) -------------------------------------------------
  if (do_s6 && sh.phase == 0 && h->t2sq_algorithm == 5) {
    plan_s6_n5(c, in, s6, XoT, XvT, YoT, YvT);
  } else if (do_s6 && local) {
    const i64 m0 = ar.mark();
    const i64 NPp = pad_to(NP, thc::TP_RT);
    // line 1: A3[Q][i][a] = sum_S Z[Q,S] Xo[i,S] Xv[a,S].  It only feeds lines 4-5 at the start of a row block.  While it
    // is small it stays resident; at paper scale (22.5 GB at config 4) it is rebuilt for every row block in the memory
    // that the I-chunk buffers reuse afterwards (+2 NP^2 o v flop per block, ~2 % of the evaluation, for 22 GB more H).
    const bool a3_resident = NP * ov * 8 <= ((i64)4 << 30) || Pe - Pb <= h->bX;
    auto build_A3 = [&](double* A3) {
      const i64 bA = std::max<i64>(1, std::min<i64>(NP, ((i64)1 << 28) / (o * NP)));      // <= 2 GB of scaled factors at a time
      for (i64 P0 = 0; P0 < NP; P0 += bA) {
        const i64 npb = std::min<i64>(bA, NP - P0), m1 = ar.mark();
        double* ZX = ar.alloc(npb * o * NP);
        c.rowscale(in.Xo, NP, in.Z + P0 * NP, NP, nullptr, 1.0, ZX, npb, o, NP);
        c.gemm(Gemm(ZX, NP, 'K', in.Xv, NP, 'K', A3 + P0 * ov, v, npb * o, v, NP));
        ar.release(m1);
      }
    };
    double* A3r = nullptr;
    if (a3_resident) { A3r = ar.alloc(NP * ov); build_A3(A3r); }
    for (i64 P0 = Pb; P0 < Pe; P0 += h->bX) {                // this rank's rows of sigma6
      const i64 npb = std::min<i64>(h->bX, Pe - P0), m1 = ar.mark();
      const i64 bXp = pad_to(npb, thc::TP_PT);
      // lines 4-5: Cc[p][(q,i)] = sum_a Xv[a,P0+p] A3[q][i][a] ;  Dd[p][(q,a)] = sum_i Xo[i,P0+p] A3[q][i][a]
      double *Cc = ar.alloc(npb * NP * o), *Dd = ar.alloc(npb * NP * v), *H = ar.alloc(bXp * NPp * NPp);
      {
        const i64 m3 = ar.mark();
        double* A3 = A3r;
        if (!a3_resident) { A3 = ar.alloc(NP * ov); build_A3(A3); }
        c.gemm(Gemm(XvT + P0 * v, v, 'K', A3, v, 'K', Cc, NP * o, npb, NP * o, v));
        c.gemm(Gemm(XoT + P0 * o, o, 'K', A3, v, 'N', Dd, NP * v, npb, v, o).batch(NP, 0, ov, v));
        ar.release(m3);
      }
      bool first = true;
      for (i64 I0 = 0; I0 < NX; I0 += h->bI) {
        const i64 ni = std::min<i64>(h->bI, NX - I0), m2 = ar.mark();
        // line 2/7: BI[I][i][a] = sum_J V[I,J] Yo[i,J] Yv[a,J]
        double *VY = ar.alloc(ni * o * NX), *BI = ar.alloc(ni * ov), *GXT = ar.alloc(ni * NP * o), *Gt = ar.alloc(ni * NPp * NPp);
        double *Eb = ar.alloc(ni * bXp * NPp), *Fb = ar.alloc(ni * bXp * NPp);
        c.rowscale(Yo, NX, in.V + I0 * NX, NX, nullptr, 1.0, VY, ni, o, NX);
        c.gemm(Gemm(VY, NX, 'K', Yv, NX, 'K', BI, v, ni * o, v, NX));
        // line 10: G_I[q][r] = sum_ia Xo[i,q] Xv[a,r] BI[I][i][a]
        c.gemm(Gemm(XvT, v, 'K', BI, v, 'K', GXT, o, NP, o, v).batch(ni, 0, ov, NP * o));
        // (line 11 reads the mirrored half G_I[r][q] from the same array: no transposed copy)
        c.gemm(Gemm(XoT, o, 'K', GXT, o, 'K', Gt, NPp, NP, NP, o).batch(ni, 0, NP * o, NPp * NPp));
        // lines 8-9: E_I[p][q] = sum_i Cc[p][(q,i)] Yo[i,I] ;  F_I[p][r] = sum_a Dd[p][(r,a)] Yv[a,I]
        c.gemm(Gemm(YoT + I0 * o, o, 'K', Cc, o, 'K', Eb, bXp * NPp, ni, NP, o).batch(npb, 0, NP * o, NPp));
        c.gemm(Gemm(YvT + I0 * v, v, 'K', Dd, v, 'K', Fb, bXp * NPp, ni, NP, v).batch(npb, 0, NP * v, NPp));
        // line 11
        c.triple_product(Eb, Fb, Gt, H, ni, bXp, NPp, first ? 0 : 1);
        first = false;
        ar.release(m2);
      }
      // lines 14-15: I^P_ia = sum_QR Xo[i,R] Xv[a,Q] H[P][Q][R] ;  s6[P][S] = sum_ia Xo[i,S] Xv[a,S] I^P_ia
      double *HT1 = ar.alloc(npb * NP * o), *Iia = ar.alloc(npb * ov), *IX = ar.alloc(npb * o * NP);
      c.gemm(Gemm(H, NPp, 'K', in.Xo, NP, 'K', HT1, o, NP, o, NP).batch(npb, NPp * NPp, 0, NP * o));
      c.gemm(Gemm(HT1, o, 'M', in.Xv, NP, 'K', Iia, v, o, v, NP).batch(npb, NP * o, 0, ov));
      c.gemm(Gemm(Iia, v, 'K', XvT, v, 'K', IX, NP, npb * o, NP, v));
      c.coldot(in.Xo, NP, IX, o * NP, NP, s6 + P0 * NP, NP, npb, NP, o);
      ar.release(m1);
    }
    ar.release(m0);
  } else if (sh.phase == 0) {
    c.fill(s6, NP2, 0.0);
  }

  // ---- Omega I, J: sigma_ia = F^_ai + sum_kc (2 t_ik^ac - t_ik^ca) F^_kc   (Eq.42 l.295; Alg.10 l.845-876) ----------------
  if (t1) {
    const i64 m0 = ar.mark();
    double *AX = ar.alloc(o * NP), *BB = ar.alloc(NP2), *dB = ar.alloc(NP), *Cx = ar.alloc(NP), *FX = ar.alloc(o * NP), *G = ar.alloc(o * NP);
    c.gemm(Gemm(F_ov, v, 'K', XvT, v, 'K', AX, NP, o, NP, v));                   // line 1: A_i^X = sum_a F^_ia y_a^X
    c.gemm(Gemm(XoT, o, 'K', AX, NP, 'N', BB, NP, NP, NP, o));                   // line 2: B^{XY} = sum_i y_i^X A_i^Y
    c.diag(BB, dB, NP);
    c.gemm(Gemm(dB, NP, 'K', in.Z, NP, 'K', Cx, NP, 1, NP, NP));                 // line 3: C^X = sum_Y T^{XY} B^{YY}
    c.hadamard(in.Z, BB, BB, NP2);                                               // line 6: E = T .* B
    c.gemm(Gemm(in.Xo, NP, 'K', BB, NP, 'K', FX, NP, o, NP, NP));                // line 7: F_i^X = sum_Y y_i^Y E^{XY}
    c.rowscale(in.Xo, NP, Cx, NP, nullptr, 2.0, G, 1, o, NP);                    // lines 4-5, 8: (2 y_i^X C^X - F_i^X) y_a^X
    c.axpby(G, FX, 1.0, -1.0, G, o * NP);
    c.copy(F_voT, sigIJ, ov);                                                    // line 10: + F^_ai
    c.gemm(Gemm(G, NP, 'K', in.Xv, NP, 'K', sigIJ, v, o, v, NP).ab(1.0, 1.0));
    if (out.sigma) c.axpby(sigGH, sigIJ, 1.0, 1.0, out.sigma, ov);
    ar.release(m0);
  }

  // ---- H11 ---------------------------------------------------------------------------------------------------------
  if (out.R) c.sum6(term, out.R, NP2);
}

// Correlation energy, factorised (R7):  E = sum_L [ 2 a^L . Z a^L - sum_PQ Z_PQ E^L_PQ E^L_QP ],
// a^L, E^L as in Alg.8 lines 5-6 (l.788-790).  Result in E_dev[0] (device).
void plan_energy(Ctx& c, const double* Xo, const double* Xv, const double* Z, const double* B_ov, double* E_dev,
                 i64 NL_local = -1) {
  thc_handle* h = c.h;
  thc::Arena& ar = c.ar;
  const i64 o = h->o, v = h->v, NL = NL_local >= 0 ? NL_local : h->NL, NP = h->NP, NP2 = NP * NP, ov = o * v;
  if (NL == 0) { c.fill(E_dev, 1, 0.0); return; }          // a rank without Cholesky vectors contributes nothing
  const i64 nblk = (NL + h->bL - 1) / h->bL;
  double *XoT = ar.alloc(NP * o), *XvT = ar.alloc(NP * v), *Aa = ar.alloc(NL * NP), *ZA = ar.alloc(NL * NP);
  double* Eblk = ar.alloc(nblk);
  c.transpose(Xo, XoT, o, NP);
  c.transpose(Xv, XvT, v, NP);
  i64 blk = 0;
  for (i64 L0 = 0; L0 < NL; L0 += h->bL, blk++) {
    const i64 nl = std::min<i64>(h->bL, NL - L0), m0 = ar.mark();
    double *TT = ar.alloc(NP * nl * o), *El = ar.alloc(nl * NP2);
    const i64 nz = c.zee_blocks(NP, nl);
    double* part = ar.alloc(nz);
    c.gemm(Gemm(XvT, v, 'K', B_ov + L0 * ov, v, 'K', TT, nl * o, NP, nl * o, v));
    c.rowdot(XoT, o, TT, o, nl * o, Aa + L0 * NP, NP, nl, NP, o);
    c.gemm(Gemm(XoT, o, 'K', TT, nl * o, 'K', El, NP, NP, NP, o).batch(nl, 0, o, NP2));
    c.zee_partial(Z, El, NP, nl, part);
    c.final_sum(part, nz, -1.0, nullptr, 0, 0.0, Eblk + blk, 0);
    ar.release(m0);
  }
  c.gemm(Gemm(Aa, NP, 'K', Z, NP, 'K', ZA, NP, NL, NP, NP));
  const i64 nd = c.dot_blocks(NL * NP);
  double* part2 = ar.alloc(nd);
  c.dot_partial(Aa, ZA, NL * NP, part2);
  c.final_sum(Eblk, nblk, 1.0, part2, nd, 2.0, E_dev, 0);
}

// ---- second workload ---------------------------------------------------------------------------------
// MP2 one-particle density matrix from THC-factorised doubles, Appendix II (l.375-415): D_oo of Eq.47, D_vv of
// Eq.48 in the O(N^4) factorisation of Eqs.51-56.  Coulomb-like parts (Eqs.53-54) are five NP^3 GEMMs and Hadamards.  The
// exchange-like parts run over blocks of occupied orbitals i, every step one (batched) DMMA GEMM:
//   Eq.55 as printed, innermost parenthesis first, with the Hadamards by o^{XZ} and the final v^{XY} sum as GEMM epilogues
//   and a row-dot;
//   Eq.56 with the o^{WZ} = sum_i y_i^W y_i^Z that closes its index cycle expanded last instead of first (the printed
//   order forms a v x NP x NP intermediate per virtual a: v NP^3 flop; summing over i last shares M_i with Eq.55 and
//   costs o NP^3):  D_ab -= 2 sum_i sum_X M_i[a][X] sum_Y o^{XY} (sum_Z y_i^Z v^{XZ} T^{YZ}) y_b^Y.
void plan_mp2_density(Ctx& c, const double* Xo, const double* Xv, const double* Z, double* D_oo, double* D_vv) {
  thc_handle* h = c.h;
  thc::Arena& ar = c.ar;
  const i64 o = h->o, v = h->v, NP = h->NP, NP2 = NP * NP, m0 = ar.mark();
  double *omat = ar.alloc(NP2), *vmat = ar.alloc(NP2), *ovm = ar.alloc(NP2), *C1 = ar.alloc(NP2), *Km = ar.alloc(NP2);
  double *tmpo = ar.alloc(o * NP), *tmpv = ar.alloc(v * NP);
  c.gemm(Gemm(Xo, NP, 'M', Xo, NP, 'N', omat, NP, NP, NP, o));                    // Eq.51
  c.gemm(Gemm(Xv, NP, 'M', Xv, NP, 'N', vmat, NP, NP, NP, v));                    // Eq.52
  c.hadamard(omat, vmat, ovm, NP2);
  c.gemm(Gemm(ovm, NP, 'K', Z, NP, 'K', C1, NP, NP, NP, NP));                     // sum_Z (o v)^{XZ} T^{YZ}
  c.gemm(Gemm(Z, NP, 'K', C1, NP, 'N', Km, NP, NP, NP, NP));                      // K^{WY} = sum_X T^{WX} ( . )
  c.hadamard(vmat, Km, C1, NP2);                                                  // Eq.53
  c.gemm(Gemm(Xo, NP, 'K', C1, NP, 'N', tmpo, NP, o, NP, NP));
  c.gemm(Gemm(tmpo, NP, 'K', Xo, NP, 'K', D_oo, o, o, o, NP).ab(-4.0, 0.0));
  c.hadamard(omat, Km, C1, NP2);                                                  // Eq.54
  c.gemm(Gemm(Xv, NP, 'K', C1, NP, 'N', tmpv, NP, v, NP, NP));
  c.gemm(Gemm(tmpv, NP, 'K', Xv, NP, 'K', D_vv, v, v, v, NP).ab(4.0, 0.0));
  const i64 per = 8 * (3 * v * NP + 2 * NP2 + NP);
  const i64 bi = std::max<i64>(1, std::min<i64>(o, ((i64)256 << 20) / per));      // 256 MB of per-block intermediates
  for (i64 i0 = 0; i0 < o; i0 += bi) {
    const i64 ni = std::min<i64>(bi, o - i0), m1 = ar.mark();
    double *Ai = ar.alloc(ni * v * NP), *Mi = ar.alloc(ni * v * NP), *Ni = ar.alloc(ni * NP2), *Ut = ar.alloc(ni * NP2);
    double *w = ar.alloc(ni * NP), *Hb = ar.alloc(ni * NP * v);
    c.rowscale(Xv, NP, Xo + i0 * NP, NP, nullptr, 1.0, Ai, ni, v, NP);                                        // y_i^W y_a^W
    c.gemm(Gemm(Ai, NP, 'K', Z, NP, 'N', Mi, NP, ni * v, NP, NP));                                           // M_i[a][X] = sum_W T^{WX} ( . )
    // Eq.55: N_i[Z][X] = o^{XZ} sum_a y_a^Z M_i[a][X];  Ut_i[Y][Z] = sum_X v^{XY} N_i[Z][X];  w_i[Y] = sum_Z T^{YZ} Ut_i[Y][Z]
    c.gemm(Gemm(Xv, NP, 'M', Mi, NP, 'N', Ni, NP, NP, NP, v).batch(ni, 0, v * NP, NP2).aux(omat, NP, 0));
    c.gemm(Gemm(vmat, NP, 'K', Ni, NP, 'K', Ut, NP, NP, NP, NP).batch(ni, 0, NP2, NP2));
    c.rowdot(Z, NP, Ut, NP2, NP, w, NP, ni, NP, NP);
    c.gemm(Gemm(w, NP, 'K', Xo, NP, 'K', D_oo + i0 * o, o, ni, o, NP).ab(2.0, 1.0));                          // sum_Y y_j^Y ( . )
    // Eq.56: Vi[X][Z] = v^{XZ} y_i^Z;  G_i[X][Y] = o^{XY} sum_Z Vi[X][Z] T^{YZ};  H_i[X][b] = sum_Y G_i[X][Y] y_b^Y
    c.rowscale(vmat, NP, Xo + i0 * NP, NP, nullptr, 1.0, Ni, ni, NP, NP);
    c.gemm(Gemm(Ni, NP, 'K', Z, NP, 'K', Ut, NP, NP, NP, NP).batch(ni, NP2, 0, NP2).aux(omat, NP, 0));
    c.gemm(Gemm(Ut, NP, 'K', Xv, NP, 'K', Hb, v, ni * NP, v, NP));
    c.gemm(Gemm(Mi, NP, 'K', Hb, v, 'N', D_vv, v, v, v, NP).kbatch(ni, v * NP, NP * v).ab(-2.0, 1.0));        // sum_i sum_X M_i[a][X] H_i[X][b]
    ar.release(m1);
  }
  ar.release(m0);
}

// One ALS factor update of a CP factorisation, Appendix I (l.355-373): S of Eq.45 (two Gram GEMMs, the Hadamard
// product in the second one's epilogue), R of Eq.46 as ONE DMMA GEMM of the unfolded array with the Khatri-Rao product
// KR[(j,k)][n] = Y_j^n Z_k^n, formed in blocks of j so that no array larger than the block is ever held (the paper
// avoids the 3-index intermediate with a custom kernel; here the block is bounded and the flops run on the tensor
// pipe), then `iters` PCG iterations on all rows at once: S p for every row is one GEMM, the rest of an iteration one
// kernel with a warp per row.
void plan_als_update(Ctx& c, i64 I, i64 J, i64 K, i64 N, const double* A, const double* Y, const double* Zf, double* X, int iters,
                     double* rnorm2) {
  thc::Arena& ar = c.ar;
  const i64 m0 = ar.mark();
  double *YtY = ar.alloc(N * N), *S = ar.alloc(N * N), *d = ar.alloc(N);
  double *R = ar.alloc(I * N), *P = ar.alloc(I * N), *SP = ar.alloc(I * N), *rz = ar.alloc(I);
  c.gemm(Gemm(Y, N, 'M', Y, N, 'N', YtY, N, N, N, J));
  c.gemm(Gemm(Zf, N, 'M', Zf, N, 'N', S, N, N, N, K).aux(YtY, N, 0));                  // Eq.45
  c.diag(S, d, N);
  const i64 bj = std::max<i64>(1, std::min<i64>(J, ((i64)64 << 20) / (8 * K * N)));      // 64 MB Khatri-Rao blocks
  for (i64 j0 = 0; j0 < J; j0 += bj) {
    const i64 nj = std::min<i64>(bj, J - j0), m1 = ar.mark();
    double* KR = ar.alloc(nj * K * N);
    c.rowscale(Zf, N, Y + j0 * N, N, nullptr, 1.0, KR, nj, K, N);                      // KR[(j,k)][n] = Z_k^n Y_j^n
    c.gemm(Gemm(A + j0 * K, J * K, 'K', KR, N, 'N', R, N, I, N, nj * K).ab(1.0, j0 ? 1.0 : 0.0));   // Eq.46
    ar.release(m1);
  }
  c.gemm(Gemm(X, N, 'K', S, N, 'K', R, N, I, N, N).ab(-1.0, 1.0));                    // r = R - X S   (S symmetric)
  c.pcg_init(R, d, P, rz, I, N);
  for (int it = 0; it < iters; it++) {
    c.gemm(Gemm(P, N, 'K', S, N, 'K', SP, N, I, N, N));
    c.pcg_iter(X, R, P, SP, d, rz, I, N);
  }
  if (rnorm2) c.rowdot(R, N, R, 0, N, rnorm2, I, 1, I, N);
  ar.release(m0);
}

// ---- dry runs: workspace sizes for the three entry points ------------------------------------------------------------
struct Need { i64 arena_bytes, splitk_doubles; i64 total() const { return arena_bytes + (splitk_doubles * 8 + 255) / 256 * 256 + 256; } };

Need dry_residual(thc_handle* h, bool with_t1 = false) {
  Ctx c{h}; c.dry = true; c.ar.dry = true;
  Inputs in{}; Outputs out{};
  if (with_t1) in.t1 = reinterpret_cast<const double*>(static_cast<uintptr_t>(256));     // only its non-nullness is used
  plan_residual(c, in, out);
  return Need{c.ar.peak, c.splitk_need};
}
Need dry_energy(thc_handle* h) {
  Ctx c{h}; c.dry = true; c.ar.dry = true;
  double* e = c.ar.alloc(1);
  plan_energy(c, nullptr, nullptr, nullptr, nullptr, e);
  return Need{c.ar.peak, c.splitk_need};
}
i64 input_doubles(const thc_handle* h, i64 sizes[9]) {
  const i64 o = h->o, v = h->v, NL = h->NL, NP = h->NP, NX = h->NX;
  const i64 s[9] = {o * NP, v * NP, NP * NP, NL * o * v, NL * o * o, NL * v * v, (o + v) * NX, NX * NX, o + v};
  i64 tot = 0;
  for (int k = 0; k < 9; k++) {
    sizes[k] = (k == 5 && h->bvv_mode != THC_BVV_DEVICE) ? 0 : s[k];     // a streamed B_vv is never staged as a whole
    tot += (sizes[k] * 8 + 255) / 256 * 256;
  }
  return tot;   // bytes
}
i64 need_device(thc_handle* h) { return std::max<i64>(dry_residual(h).total(), dry_energy(h).total()); }
i64 need_host(thc_handle* h) {
  i64 sz[9];
  Need r = dry_residual(h), e = dry_energy(h);
  i64 staging = input_doubles(h, sz) + (h->NP * h->NP * 8 + 255) / 256 * 256 + 256;
  return staging + std::max<i64>(r.total(), e.total());
}

bool bad_ptr(const void* p) { return p == nullptr || (reinterpret_cast<uintptr_t>(p) & 7) != 0; }

// Make sure a workspace of `bytes` exists (library-owned unless the caller provided one).
int ensure_workspace(thc_handle* h, i64 bytes) {
  if (h->ws && h->ws_bytes >= bytes) return THC_OK;
  if (h->ws && !h->ws_owned) return THC_ERR_NO_MEMORY;     // caller's buffer is too small
  if (h->ws) { cudaStreamSynchronize(h->stream); cudaFree(h->ws); h->ws = nullptr; h->ws_bytes = 0; }
  void* p = nullptr;
  cudaError_t e = cudaMalloc(&p, (size_t)bytes);
  if (e != cudaSuccess) { h->last_cuda = (int)e; cudaGetLastError(); return THC_ERR_NO_MEMORY; }
  h->ws = p; h->ws_bytes = bytes; h->ws_owned = true;
  return THC_OK;
}

// Real-run context over [base, base + bytes): split-K scratch first, arena after it.
int make_ctx(Ctx& c, thc_handle* h, char* base, i64 bytes, const Need& need) {
  if (need.total() > bytes) return THC_ERR_NO_MEMORY;
  c.h = h; c.dry = false;
  uintptr_t b = (reinterpret_cast<uintptr_t>(base) + 255) / 256 * 256;
  c.splitk = reinterpret_cast<double*>(b);
  c.splitk_cap = need.splitk_doubles;
  i64 sk = (need.splitk_doubles * 8 + 255) / 256 * 256;
  c.ar.base = reinterpret_cast<char*>(b) + sk;
  c.ar.cap = bytes - sk - (i64)(b - reinterpret_cast<uintptr_t>(base));
  c.ar.dry = false;
  return THC_OK;
}

// thc_options.check_symmetry (debug): Z, V, every B^L_oo and -- when resident -- every B^L_vv must be symmetric to 1e-12
// of their largest element, because the plan evaluates symmetric products on one triangle only (thc.h).  One pass over
// HBM and one host synchronisation; NL_local Cholesky vectors are present.
int check_symmetric(thc_handle* h, const Inputs& in, i64 NL_local) {
  if (!h->sym_scratch) {
    void* p = nullptr;
    cudaError_t e = cudaMalloc(&p, 8 * sizeof(double));
    if (e != cudaSuccess) { h->last_cuda = (int)e; cudaGetLastError(); return THC_ERR_NO_MEMORY; }
    h->sym_scratch = static_cast<double*>(p);
  }
  cudaError_t e = cudaMemsetAsync(h->sym_scratch, 0, 8 * sizeof(double), h->stream);
  if (e != cudaSuccess) { h->last_cuda = (int)e; return THC_ERR_CUDA; }
  unsigned long long* out = reinterpret_cast<unsigned long long*>(h->sym_scratch);
  struct Item { const double* A; i64 n, nb; } items[4] = {
      {in.Z, h->NP, 1}, {in.V, h->NX, 1}, {in.B_oo, h->o, NL_local},
      {h->bvv_mode == THC_BVV_DEVICE ? static_cast<const double*>(in.B_vv) : nullptr, h->v, NL_local}};
  for (int k = 0; k < 4; k++) {
    if (!items[k].A || items[k].nb <= 0) continue;
    const i64 total = items[k].nb * items[k].n * items[k].n;
    const int blocks = (int)std::max<i64>(1, std::min<i64>((total + 255) / 256, (i64)h->sms * 16));
    thc::asym_max_kernel<<<blocks, 256, 0, h->stream>>>(items[k].A, (int)items[k].n, items[k].nb, out + 2 * k);
    h->launches++;
  }
  double res[8];
  e = cudaMemcpyAsync(res, h->sym_scratch, sizeof res, cudaMemcpyDeviceToHost, h->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
  if (e != cudaSuccess) { h->last_cuda = (int)e; return THC_ERR_CUDA; }
  for (int k = 0; k < 4; k++)
    if (res[2 * k] > 1e-12 * res[2 * k + 1]) return THC_ERR_INVALID_ARG;
  return THC_OK;
}

struct DeviceGuard {
  int prev = -1; bool ok = true;
  explicit DeviceGuard(int dev) { if (cudaGetDevice(&prev) != cudaSuccess) ok = false; else if (prev != dev) ok = cudaSetDevice(dev) == cudaSuccess; }
  ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

int run_residual(thc_handle* h, char* base, i64 bytes, const Inputs& in, const Outputs& out, const Shard& sh = Shard()) {
  Need need = dry_residual(h, in.t1 != nullptr && sh.phase == 0);
  Ctx c{h};
  int st = make_ctx(c, h, base, bytes, need);
  if (st != THC_OK) return st;
  plan_residual(c, in, out, sh);
  if (c.ar.overflow) return THC_ERR_NO_MEMORY;
  return c.status;
}

// Run `body` (which enqueues one evaluation on h->stream) either directly or through the cached CUDA graph of `slot`
// (thc_handle::GraphSlot).  `key` = every pointer the evaluation depends on.
template <typename Body>
int run_maybe_graphed(thc_handle* h, int slot, std::vector<uintptr_t> key, Body body) {
  const bool eligible = h->graph_on && h->bvv_mode == THC_BVV_DEVICE && h->prof_mask == 0;
  if (!eligible) return body();
  key.push_back(reinterpret_cast<uintptr_t>(h->ws));
  key.push_back((uintptr_t)h->ws_bytes);
  key.push_back(reinterpret_cast<uintptr_t>(h->stream));
  thc_handle::GraphSlot& g = h->graph[slot];
  if (g.key != key) {
    if (g.exec) { cudaGraphExecDestroy(g.exec); g.exec = nullptr; }
    g.key = key;
    g.seen = 0;
  }
  g.seen++;
  if (g.seen == 1) return body();                       // eager: one-time opt-ins, work lists, descriptor entry point
  if (!g.exec) {
    if (!h->cap_stream && cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking) != cudaSuccess) {
      cudaGetLastError();
      h->graph_on = false;
      return body();
    }
    cudaStream_t user = h->stream;
    const int64_t l0 = h->launches;
    h->stream = h->cap_stream;
    cudaGraph_t graph = nullptr;
    cudaError_t e = cudaStreamBeginCapture(h->cap_stream, cudaStreamCaptureModeThreadLocal);
    int st = THC_OK;
    if (e == cudaSuccess) {
      st = body();
      e = cudaStreamEndCapture(h->cap_stream, &graph);
    }
    h->stream = user;
    if (e == cudaSuccess && st == THC_OK) e = cudaGraphInstantiate(&g.exec, graph, 0);
    if (graph) cudaGraphDestroy(graph);
    if (e != cudaSuccess || st != THC_OK || !g.exec) {  // capture not possible here: fall back to plain launches for good
      cudaGetLastError();
      g.exec = nullptr;
      h->graph_on = false;
      h->launches = l0;
      return body();
    }
    g.launches = h->launches - l0;
    h->launches = l0;
  }
  cudaError_t e = cudaGraphLaunch(g.exec, h->stream);
  if (e != cudaSuccess) { h->last_cuda = (int)e; return THC_ERR_CUDA; }
  h->launches += g.launches;
  return THC_OK;
}
int run_energy(thc_handle* h, char* base, i64 bytes, const double* Xo, const double* Xv, const double* Z, const double* B_ov,
               double* E_host, double* E_dev, i64 NL_local = -1) {
  Need need = dry_energy(h);
  Ctx c{h};
  int st = make_ctx(c, h, base, bytes, need);
  if (st != THC_OK) return st;
  double* e = c.ar.alloc(1);
  plan_energy(c, Xo, Xv, Z, B_ov, E_dev ? E_dev : e, NL_local);
  if (c.ar.overflow) return THC_ERR_NO_MEMORY;
  if (c.status != THC_OK) return c.status;
  if (E_host) {
    c.check(cudaMemcpyAsync(E_host, E_dev ? E_dev : e, sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    c.check(cudaStreamSynchronize(h->stream));
  }
  return c.status;
}

}  // namespace

// =====================================================================================================================
// C ABI
// =====================================================================================================================
extern "C" {

int thc_setup(thc_handle** hp, int64_t o, int64_t v, int64_t NL, int64_t NP, int64_t NX, const thc_options* opt) {
  if (!hp) return THC_ERR_INVALID_ARG;
  *hp = nullptr;
  if (o <= 0 || v <= 0 || NL <= 0 || NP <= 0 || NX <= 0) return THC_ERR_INVALID_ARG;
  if (opt && (opt->bvv_mode < 0 || opt->bvv_mode > 2 || opt->use_graph < -1 || opt->use_graph > 1 ||
              (opt->t2sq_algorithm != 0 && opt->t2sq_algorithm != 4 && opt->t2sq_algorithm != 5)))
    return THC_ERR_INVALID_ARG;
  if (opt && (opt->bL < 0 || opt->bP7 < 0 || opt->bX < 0 || opt->bI < 0 || opt->workspace_bytes_max < 0)) return THC_ERR_INVALID_ARG;
  const int64_t lim = (int64_t)1 << 31;
  if (o >= lim || v >= lim || NL >= lim || NP >= lim || NX >= lim) return THC_ERR_OVERFLOW;
  // largest single buffers must stay below 2^60 bytes and GEMM extents below 2^31
  const long double big = (long double)NL * v * v;
  if (big * 8 > 1e18L || (long double)NP * NP * std::max<i64>(o, v) > 9e18L) return THC_ERR_OVERFLOW;
  if ((long double)NP * o * 64 >= (long double)lim || (long double)NX * NX >= 9e18L) return THC_ERR_OVERFLOW;

  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); return THC_ERR_NO_DEVICE; }
  int dev = (opt && opt->device >= 0) ? opt->device : -1;
  if (dev < 0 && cudaGetDevice(&dev) != cudaSuccess) return THC_ERR_NO_DEVICE;
  if (dev >= ndev) return THC_ERR_INVALID_ARG;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return THC_ERR_NO_DEVICE;
  if (prop.major != 10) return THC_ERR_NO_DEVICE;     // sm_100a binary only

  thc_handle* h = new (std::nothrow) thc_handle();
  if (!h) return THC_ERR_NO_MEMORY;
  h->o = o; h->v = v; h->NL = NL; h->NP = NP; h->NX = NX;
  h->term_mask = opt ? (opt->term_mask & THC_TERM_ALL) : 0;
  h->device = dev; h->sms = prop.multiProcessorCount;
  h->stream = nullptr; h->ws = nullptr; h->ws_bytes = 0; h->ws_owned = false;
  h->launches = 0; h->last_cuda = 0; h->smem_configured = false;
  h->gemm_smem_mask = 0; h->ring_smem_mask = 0; h->tma_min_flop = (opt && opt->tma_min_flop) ? (double)opt->tma_min_flop : 2e8;
  h->check_symmetry = opt ? opt->check_symmetry : 0; h->sym_scratch = nullptr;
  {
    // Alg.6 vs Alg.4+5 ("ideally one would..."): leading flop counts over measured rates (line 11 ~17
    // TFLOP/s, GEMMs of a G pass ~30, the many small batched products of Alg.4/5 ~12: 7.5 at config 1, 14 at config 2)
    // plus ~5 us per launch (Alg.4/5 loop over i and a).  Measured sigma6 times, Alg.6 / Alg.4+5: config 0 0.26 / 0.92 ms,
    // config 1 7.3 / 20.3 ms, config 2 0.64 / 2.36 s -- on B200 the crossover the paper saw on V100 is below config 0.
    const double fo = (double)o, fv = (double)v, fP = (double)NP, fX = (double)NX;
    const double t4 = 5 * fX * fP * fP * fP / 17e12 + (2 * (fo + fv) * fP * fP * fX + fX * (2 * fo * fv * fP + 2 * fo * fP * fP + 2 * fo * fv * fX)) / 30e12 + 5e-6 * 20;
    const double t5 = (fo * fo * (2 * fv * fX * fX + 2 * fo * fX * fX + 2 * fo * fP * fP + 4 * fv * fP * fP + 2 * fv * fv * (fX + 2 * fP)) +
                       fo * fv * (4 * fo * fX * fX + 6 * fo * fP * fP + 2 * fo * fv * (fX + 2 * fP))) / 12e12 + 5e-6 * (3 * (fo + fv) + 30);
    const int want = opt ? opt->t2sq_algorithm : 0;
    const bool n5_fits = (double)o * NX * NX * 8 < 8e9;
    h->t2sq_algorithm = want ? want : ((t5 < t4 && n5_fits) ? 5 : 4);
  }
  h->prof_mask = 0; h->prof_used = 0; h->prof_done = 0; h->encode_tiled = nullptr;
  h->tp_gate = true;
  h->cap_stream = nullptr;
  {
    const int ug = opt ? opt->use_graph : -1;
    const bool resident = (opt ? opt->bvv_mode : THC_BVV_DEVICE) == THC_BVV_DEVICE;
    h->graph_on = resident && (ug == 1 || (ug == -1 && thc_algorithmic_flops(h) < 2e10));   // auto: launch-bound shapes only
  }
  h->bvv_mode = opt ? opt->bvv_mode : THC_BVV_DEVICE; h->copy_stream = nullptr; h->copy_ready = false;

  // block sizes: defaults, then shrink until the plan fits the cap
  h->bL = std::min<int64_t>(NL, (opt && opt->bL) ? opt->bL : 512);    // long L-blocks: few, large GEMMs (shrunk below if HBM is short)
  const int64_t p7_auto = o <= 64 ? std::max<int64_t>(1, ((int64_t)2 << 30) / (NX * (o + v) * 8 + 1))
                                  : std::max<int64_t>(1, ((int64_t)8 << 30) / (NX * NX * 8));   // E .* V is materialised
  h->bP7 = std::min<int64_t>(NP, (opt && opt->bP7) ? opt->bP7 : p7_auto);
  h->bX = std::min<int64_t>(pad_to(NP, 16), (opt && opt->bX) ? pad_to(opt->bX, 16) : pad_to(NP, 16));
  h->bI = std::min<int64_t>(NX, (opt && opt->bI) ? opt->bI : 1024);   // long I loops amortise the H read-modify-write
  int64_t cap = opt ? opt->workspace_bytes_max : 0;
  if (cap == 0) {
    DeviceGuard g(dev);
    size_t fr = 0, tot = 0;
    if (!g.ok || cudaMemGetInfo(&fr, &tot) != cudaSuccess) { delete h; return THC_ERR_CUDA; }
    // the workspace is the only large allocation the library makes; the T2^2 phases at paper scale need every GB
    cap = (int64_t)(0.92 * (double)fr);
  }
  const bool fix_bX = opt && opt->bX, fix_bI = opt && opt->bI, fix_bP7 = opt && opt->bP7, fix_bL = opt && opt->bL;
  {
    // stage A: the L-block loop and the T2^2 phases reuse the same arena, so first find the largest bL whose own phase
    // fits (the other block sizes at their minimum), then size the rest with bL fixed
    const int64_t sX = h->bX, sP = h->bP7, sI = h->bI;
    if (!fix_bX) h->bX = 16;
    if (!fix_bP7) h->bP7 = 1;
    if (!fix_bI) h->bI = std::min<int64_t>(NX, 16);
    while (!fix_bL && h->bL > 1 && need_device(h) > cap) h->bL = h->bL / 2;
    // stage B: the Alg.7 phase on its own
    h->bP7 = sP;
    while (!fix_bP7 && h->bP7 > 1 && need_device(h) > cap) h->bP7 = h->bP7 / 2;
    // stage C: Alg.6.  H[bX][NPp][NPp] and the G_I chunk (bI grid points, both orientations) compete for the same
    // memory: every row block recomputes all G_I (cost ~ 1/bX), every chunk reads and rewrites H (cost ~ 1/bI).  Take
    // the (bX, bI) pair that minimises  ceil(NP/bX) * t(G pass) + ceil(NX/bI) * t(H read + write)  among those that fit.
    h->bX = sX; h->bI = sI;
    if (!fix_bX && !fix_bI && need_device(h) > cap) {
      const double fo = (double)o, fv = (double)v, fNP = (double)NP, fNX = (double)NX;
      // measured on B200 (profiles/r02_final.md, config 4): one G pass (B_ia^I, its two half-transforms, A3 rebuilt when it
      // is not resident) runs at ~30 TFLOP/s = 9.6 s; the read-modify-write of H at the end of every work item of line 11
      // is not overlapped with its FMAs and costs 6 % of a launch with 128-point chunks (17.9 vs 19.0 TFLOP/s), i.e. its
      // bytes at ~7 TB/s.
      const double t_g = (fNX * (2 * fo * fv * fNX + 2 * fo * fv * fNP + 2 * fo * fNP * fNP) +
                          (NP * o * v * 8 > ((i64)4 << 30) ? 2 * fNP * fNP * fo * fv : 0.0)) / 30e12;            // DMMA, s
      const double t_h = 16.0 * fNP * (double)pad_to(NP, 32) * (double)pad_to(NP, 32) / 7e12;            // HBM, s
      double best = 1e300; int64_t bestX = 0, bestI = 0;
      // (chunks of a multiple of 128 grid points fill the 128-row tiles of the E_I / F_I products)
      for (int64_t bi : {16, 32, 64, 128, 256, 384, 512, 640, 768, 896, 1024}) {
        if (bi > NX) break;
        h->bI = bi; h->bX = 16;
        if (need_device(h) > cap) break;
        int64_t lo = 1, hi = pad_to(NP, 16) / 16;              // largest bX = 16 * lo that fits
        while (lo < hi) {
          const int64_t mid = (lo + hi + 1) / 2;
          h->bX = 16 * mid;
          if (need_device(h) <= cap) lo = mid; else hi = mid - 1;
        }
        const int64_t bx = 16 * lo;
        const double t = std::ceil(fNP / (double)bx) * t_g + std::ceil(fNX / (double)bi) * t_h;
        if (t < best) { best = t; bestX = bx; bestI = bi; }
      }
      if (bestX) { h->bX = bestX; h->bI = bestI; } else { h->bX = sX; h->bI = sI; }
    }
  }
  for (;;) {
    h->need_bytes = need_device(h);
    if (h->need_bytes <= cap) break;
    if (!fix_bX && h->bX > 512) h->bX = pad_to(h->bX / 2, 16);
    else if (!fix_bI && h->bI > 128) h->bI = h->bI / 2;
    else if (!fix_bX && h->bX > 64) h->bX = pad_to(h->bX / 2, 16);
    else if (!fix_bP7 && h->bP7 > 1) h->bP7 = h->bP7 / 2;
    else if (!fix_bL && h->bL > 4) h->bL = h->bL / 2;
    else if (!fix_bI && h->bI > 16) h->bI = h->bI / 2;
    else if (!fix_bX && h->bX > 16) h->bX = pad_to(h->bX / 2, 16);
    else if (!fix_bL && h->bL > 1) h->bL = h->bL / 2;
    else { delete h; return THC_ERR_NO_MEMORY; }
  }
  // The work lists of Alg.6 line 11 for the row blocks of an unsharded evaluation (full block and tail) are uploaded
  // here, so that the first evaluation neither allocates nor synchronises; other shapes (shards) are built on first use.
  if (h->t2sq_algorithm != 5 && (h->term_mask == 0 || (h->term_mask & THC_TERM_S6))) {
    DeviceGuard g(dev);
    Ctx c{h};
    c.dry = false;
    const i64 NPp = pad_to(NP, thc::TP_RT), full = std::min<i64>(h->bX, NP), tail = NP % full;
    if (g.ok) {
      c.triple_items(pad_to(full, thc::TP_PT), NPp);
      if (tail) c.triple_items(pad_to(tail, thc::TP_PT), NPp);
    }
    if (!g.ok || c.status != THC_OK) { const int st = g.ok ? c.status : THC_ERR_CUDA; thc_destroy(h); return st; }
  }
  *hp = h;
  return THC_OK;
}

int thc_destroy(thc_handle* h) {
  if (!h) return THC_ERR_INVALID_ARG;
  if ((h->ws && h->ws_owned) || !h->prof_events.empty() || !h->tp_lists.empty() || h->copy_ready || h->sym_scratch ||
      h->cap_stream || h->graph[0].exec || h->graph[1].exec) {
    DeviceGuard g(h->device);
    cudaStreamSynchronize(h->stream);
    if (h->ws && h->ws_owned) cudaFree(h->ws);
    for (cudaEvent_t e : h->prof_events) cudaEventDestroy(e);
    for (auto& l : h->tp_lists) cudaFree(l.dev);
    if (h->sym_scratch) cudaFree(h->sym_scratch);
    for (auto& gs : h->graph) if (gs.exec) cudaGraphExecDestroy(gs.exec);
    if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
    if (h->copy_ready) {
      cudaStreamSynchronize(h->copy_stream);
      for (int k = 0; k < 2; k++) { cudaEventDestroy(h->ev_loaded[k]); cudaEventDestroy(h->ev_free[k]); }
      cudaEventDestroy(h->ev_start);
      cudaStreamDestroy(h->copy_stream);
    }
  }
  delete h;
  return THC_OK;
}

int64_t thc_workspace_bytes(const thc_handle* h) { return h ? h->need_bytes : (int64_t)THC_ERR_INVALID_ARG; }
int64_t thc_workspace_bytes_host(const thc_handle* h) { return h ? need_host(const_cast<thc_handle*>(h)) : (int64_t)THC_ERR_INVALID_ARG; }

int thc_set_workspace(thc_handle* h, void* device_ptr, int64_t bytes) {
  if (!h || !device_ptr || bytes <= 0) return THC_ERR_INVALID_ARG;
  if (h->ws && h->ws_owned) {
    DeviceGuard g(h->device);
    cudaStreamSynchronize(h->stream);
    cudaFree(h->ws);
  }
  h->ws = device_ptr; h->ws_bytes = bytes; h->ws_owned = false;
  return THC_OK;
}

int thc_set_stream(thc_handle* h, void* cuda_stream) {
  if (!h) return THC_ERR_INVALID_ARG;
  h->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
  return THC_OK;
}

int thc_get_blocks(const thc_handle* h, int64_t out[4]) {
  if (!h || !out) return THC_ERR_INVALID_ARG;
  out[0] = h->bL; out[1] = h->bP7; out[2] = h->bX; out[3] = h->bI;
  return THC_OK;
}

int thc_residual_terms(thc_handle* h, const double* Xo, const double* Xv, const double* Z, const double* B_ov,
                       const double* B_oo, const void* B_vv, const double* Y, const double* V, const double* eps,
                       double* R, double* const terms[6], double* xi_oo, double* xi_vv) {
  if (!h) return THC_ERR_INVALID_ARG;
  if (bad_ptr(Xo) || bad_ptr(Xv) || bad_ptr(Z) || bad_ptr(B_ov) || bad_ptr(B_oo) || bad_ptr(B_vv) || bad_ptr(Y) ||
      bad_ptr(V) || bad_ptr(eps))
    return THC_ERR_INVALID_ARG;
  Inputs in{Xo, Xv, Z, B_ov, B_oo, B_vv, Y, V, eps};
  Outputs out{};
  out.R = R;
  bool any = R != nullptr;
  for (int k = 0; k < 6; k++) { out.terms[k] = terms ? terms[k] : nullptr; any = any || out.terms[k]; }
  out.xi_oo = xi_oo; out.xi_vv = xi_vv;
  if (!any && !xi_oo && !xi_vv) return THC_ERR_INVALID_ARG;
  if ((R && bad_ptr(R)) || (xi_oo && bad_ptr(xi_oo)) || (xi_vv && bad_ptr(xi_vv))) return THC_ERR_INVALID_ARG;
  DeviceGuard g(h->device);
  if (!g.ok) return THC_ERR_CUDA;
  int st = ensure_workspace(h, h->need_bytes);
  if (st != THC_OK) return st;
  if (h->check_symmetry && (st = check_symmetric(h, in, h->NL)) != THC_OK) return st;
  std::vector<uintptr_t> key;
  for (const void* q : {(const void*)Xo, (const void*)Xv, (const void*)Z, (const void*)B_ov, (const void*)B_oo, B_vv, (const void*)Y,
                        (const void*)V, (const void*)eps, (const void*)R, (const void*)xi_oo, (const void*)xi_vv})
    key.push_back(reinterpret_cast<uintptr_t>(q));
  for (int k = 0; k < 6; k++) key.push_back(reinterpret_cast<uintptr_t>(out.terms[k]));
  return run_maybe_graphed(h, 0, key, [&] { return run_residual(h, static_cast<char*>(h->ws), h->ws_bytes, in, out); });
}

int thc_residual(thc_handle* h, const double* Xo, const double* Xv, const double* Z, const double* B_ov,
                 const double* B_oo, const void* B_vv, const double* Y, const double* V, const double* eps, double* R) {
  if (!R) return THC_ERR_INVALID_ARG;
  return thc_residual_terms(h, Xo, Xv, Z, B_ov, B_oo, B_vv, Y, V, eps, R, nullptr, nullptr, nullptr);
}

int64_t thc_workspace_bytes_t1(const thc_handle* h) {
  return h ? dry_residual(const_cast<thc_handle*>(h), true).total() : (int64_t)THC_ERR_INVALID_ARG;
}

int thc_residual_t1(thc_handle* h, const double* Xo, const double* Xv, const double* Z, const double* t1, const double* B_ov,
                    const double* B_oo, const void* B_vv, const double* Y, const double* V, const double* eps, double* R,
                    double* sigma, double* const terms[6], double* const sigma_terms[2], double* xi_oo, double* xi_vv) {
  if (!h) return THC_ERR_INVALID_ARG;
  if (bad_ptr(Xo) || bad_ptr(Xv) || bad_ptr(Z) || bad_ptr(t1) || bad_ptr(B_ov) || bad_ptr(B_oo) || bad_ptr(B_vv) || bad_ptr(Y) ||
      bad_ptr(V) || bad_ptr(eps) || bad_ptr(R) || bad_ptr(sigma) || (xi_oo && bad_ptr(xi_oo)) || (xi_vv && bad_ptr(xi_vv)))
    return THC_ERR_INVALID_ARG;
  if ((h->term_mask ? h->term_mask : THC_TERM_ALL) != THC_TERM_ALL) return THC_ERR_INVALID_ARG;     // a complete residual only
  Inputs in{Xo, Xv, Z, B_ov, B_oo, B_vv, Y, V, eps};
  in.t1 = t1;
  Outputs out{};
  out.R = R; out.sigma = sigma; out.xi_oo = xi_oo; out.xi_vv = xi_vv;
  for (int k = 0; k < 6; k++) out.terms[k] = terms ? terms[k] : nullptr;
  for (int k = 0; k < 2; k++) out.sigma_parts[k] = sigma_terms ? sigma_terms[k] : nullptr;
  DeviceGuard g(h->device);
  if (!g.ok) return THC_ERR_CUDA;
  int st = ensure_workspace(h, std::max<i64>(h->need_bytes, thc_workspace_bytes_t1(h)));
  if (st != THC_OK) return st;
  if (h->check_symmetry && (st = check_symmetric(h, in, h->NL)) != THC_OK) return st;
  return run_residual(h, static_cast<char*>(h->ws), h->ws_bytes, in, out);
}

int64_t thc_workspace_bytes_rr(const thc_handle* h, int64_t NR) {
  if (!h || NR <= 0) return (int64_t)THC_ERR_INVALID_ARG;
  auto pad = [](i64 n) { return (n * 8 + 255) / 256 * 256; };
  return h->need_bytes + 2 * pad(h->NP * h->NP) + pad(NR * h->NP) + 256;
}

int thc_residual_rr(thc_handle* h, int64_t NR, const double* tau, const double* T, const double* Xo, const double* Xv,
                    const double* B_ov, const double* B_oo, const void* B_vv, const double* Y, const double* V,
                    const double* eps, double* R_rr, double* Z_out) {
  if (!h || NR <= 0 || NR >= ((int64_t)1 << 31)) return THC_ERR_INVALID_ARG;
  if (bad_ptr(tau) || bad_ptr(T) || bad_ptr(Xo) || bad_ptr(Xv) || bad_ptr(B_ov) || bad_ptr(B_oo) || bad_ptr(B_vv) || bad_ptr(Y) ||
      bad_ptr(V) || bad_ptr(eps) || bad_ptr(R_rr) || (Z_out && bad_ptr(Z_out)))
    return THC_ERR_INVALID_ARG;
  DeviceGuard g(h->device);
  if (!g.ok) return THC_ERR_CUDA;
  int st = ensure_workspace(h, thc_workspace_bytes_rr(h, NR));
  if (st != THC_OK) return st;
  const i64 NP = h->NP;
  auto pad = [](i64 n) { return (n * 8 + 255) / 256 * 256; };
  char* p = reinterpret_cast<char*>((reinterpret_cast<uintptr_t>(h->ws) + 255) / 256 * 256);
  double* Z = reinterpret_cast<double*>(p); p += pad(NP * NP);
  double* R = reinterpret_cast<double*>(p); p += pad(NP * NP);
  double* tmp = reinterpret_cast<double*>(p); p += pad(NR * NP);
  const i64 rest = h->ws_bytes - (p - static_cast<char*>(h->ws));
  {
    // Z[W][X] = sum_PQ tau[P][W] T[P][Q] tau[Q][X]:  tmp = T tau,  Z = tau^T tmp       (Eq.22 l.178)
    Ctx c{h}; c.dry = false;
    c.gemm(Gemm(T, NR, 'K', tau, NP, 'N', tmp, NP, NR, NP, NR));
    c.gemm(Gemm(tau, NP, 'M', tmp, NP, 'N', Z, NP, NP, NP, NR));
    if (c.status != THC_OK) return c.status;
    if (Z_out) {
      cudaError_t e = cudaMemcpyAsync(Z_out, Z, (size_t)NP * NP * 8, cudaMemcpyDeviceToDevice, h->stream);
      if (e != cudaSuccess) { h->last_cuda = (int)e; return THC_ERR_CUDA; }
    }
  }
  Inputs in{Xo, Xv, Z, B_ov, B_oo, B_vv, Y, V, eps};
  Outputs out{};
  out.R = R;
  if (h->check_symmetry && (st = check_symmetric(h, in, h->NL)) != THC_OK) return st;
  st = run_residual(h, p, rest, in, out);
  if (st != THC_OK) return st;
  {
    // R_rr[P][Q] = sum_WX tau[P][W] R[W][X] tau[Q][X]:  tmp = tau R,  R_rr = tmp tau^T   (Eqs.6, 14)
    Ctx c{h}; c.dry = false;
    c.gemm(Gemm(tau, NP, 'K', R, NP, 'N', tmp, NP, NR, NP, NP));
    c.gemm(Gemm(tmp, NP, 'K', tau, NP, 'K', R_rr, NR, NR, NR, NP));
    return c.status;
  }
}

int thc_energy(thc_handle* h, const double* Xo, const double* Xv, const double* Z, const double* B_ov, double* E_host) {
  if (!h || bad_ptr(Xo) || bad_ptr(Xv) || bad_ptr(Z) || bad_ptr(B_ov) || !E_host) return THC_ERR_INVALID_ARG;
  DeviceGuard g(h->device);
  if (!g.ok) return THC_ERR_CUDA;
  int st = ensure_workspace(h, h->need_bytes);
  if (st != THC_OK) return st;
  return run_energy(h, static_cast<char*>(h->ws), h->ws_bytes, Xo, Xv, Z, B_ov, E_host, nullptr);
}

int thc_energy_device(thc_handle* h, const double* Xo, const double* Xv, const double* Z, const double* B_ov, double* E_dev) {
  if (!h || bad_ptr(Xo) || bad_ptr(Xv) || bad_ptr(Z) || bad_ptr(B_ov) || bad_ptr(E_dev)) return THC_ERR_INVALID_ARG;
  DeviceGuard g(h->device);
  if (!g.ok) return THC_ERR_CUDA;
  int st = ensure_workspace(h, h->need_bytes);
  if (st != THC_OK) return st;
  std::vector<uintptr_t> key;
  for (const void* q : {(const void*)Xo, (const void*)Xv, (const void*)Z, (const void*)B_ov, (const void*)E_dev})
    key.push_back(reinterpret_cast<uintptr_t>(q));
  return run_maybe_graphed(h, 1, key, [&] { return run_energy(h, static_cast<char*>(h->ws), h->ws_bytes, Xo, Xv, Z, B_ov, nullptr, E_dev); });
}

// ---- sharded evaluation -----------------------------------------------------------------------------
int thc_shard_range(int64_t NL, int64_t NP, int rank, int nranks, int64_t out[4]) {
  if (!out || NL <= 0 || NP <= 0 || nranks <= 0 || rank < 0 || rank >= nranks) return THC_ERR_INVALID_ARG;
  out[0] = NL * rank / nranks; out[1] = NL * (rank + 1) / nranks;          // equal contiguous Cholesky ranges (l.220)
  out[2] = NP * rank / nranks; out[3] = NP * (rank + 1) / nranks;          // equal contiguous row blocks (l.257, l.273)
  return THC_OK;
}

int64_t thc_shard_doubles(const thc_handle* h) {
  return h ? PackedLayout(h->o, h->v, h->NP, h->NX).total : (int64_t)THC_ERR_INVALID_ARG;
}

int thc_residual_shard(thc_handle* h, const double* Xo, const double* Xv, const double* Z, const double* B_ov,
                       const double* B_oo, const void* B_vv, const double* Y, const double* V, const double* eps,
                       int rank, int nranks, double* packed) {
  if (!h || bad_ptr(Xo) || bad_ptr(Xv) || bad_ptr(Z) || bad_ptr(Y) || bad_ptr(V) || bad_ptr(eps) || bad_ptr(packed))
    return THC_ERR_INVALID_ARG;
  int64_t r[4];
  int st = thc_shard_range(h->NL, h->NP, rank, nranks, r);
  if (st != THC_OK) return st;
  if (r[1] > r[0] && (bad_ptr(B_ov) || bad_ptr(B_oo) || bad_ptr(B_vv))) return THC_ERR_INVALID_ARG;
  Inputs in{Xo, Xv, Z, B_ov, B_oo, B_vv, Y, V, eps};
  Outputs out{};
  Shard sh;
  sh.phase = 1; sh.Lb = r[0]; sh.Le = r[1]; sh.Pb = r[2]; sh.Pe = r[3]; sh.packed = packed;
  DeviceGuard g(h->device);
  if (!g.ok) return THC_ERR_CUDA;
  st = ensure_workspace(h, h->need_bytes);
  if (st != THC_OK) return st;
  if (h->check_symmetry && (st = check_symmetric(h, in, r[1] - r[0])) != THC_OK) return st;
  return run_residual(h, static_cast<char*>(h->ws), h->ws_bytes, in, out, sh);
}

int thc_residual_finish(thc_handle* h, const double* Xo, const double* Xv, const double* Z, const double* Y,
                        const double* V, const double* eps, double* packed, double* R, double* const terms[6]) {
  if (!h || bad_ptr(Xo) || bad_ptr(Xv) || bad_ptr(Z) || bad_ptr(Y) || bad_ptr(V) || bad_ptr(eps) || bad_ptr(packed) ||
      bad_ptr(R))
    return THC_ERR_INVALID_ARG;
  Inputs in{Xo, Xv, Z, nullptr, nullptr, nullptr, Y, V, eps};
  Outputs out{};
  out.R = R;
  if (terms) { out.terms[2] = terms[2]; out.terms[5] = terms[5]; }     // s3, s9; the other four live in `packed`
  Shard sh;
  sh.phase = 2; sh.packed = packed;
  DeviceGuard g(h->device);
  if (!g.ok) return THC_ERR_CUDA;
  int st = ensure_workspace(h, h->need_bytes);
  if (st != THC_OK) return st;
  st = run_residual(h, static_cast<char*>(h->ws), h->ws_bytes, in, out, sh);
  if (st != THC_OK || !terms) return st;
  const PackedLayout pk(h->o, h->v, h->NP, h->NX);
  const i64 off[6] = {pk.s1, pk.s2, -1, pk.s6, pk.s7, -1};
  for (int k = 0; k < 6; k++)
    if (off[k] >= 0 && terms[k]) {
      cudaError_t e = cudaMemcpyAsync(terms[k], packed + off[k], (size_t)h->NP * h->NP * 8, cudaMemcpyDeviceToDevice, h->stream);
      if (e != cudaSuccess) { h->last_cuda = (int)e; return THC_ERR_CUDA; }
    }
  return THC_OK;
}

int thc_energy_shard(thc_handle* h, const double* Xo, const double* Xv, const double* Z, const double* B_ov, int rank,
                     int nranks, double* E_dev) {
  if (!h || bad_ptr(Xo) || bad_ptr(Xv) || bad_ptr(Z) || bad_ptr(E_dev)) return THC_ERR_INVALID_ARG;
  int64_t r[4];
  int st = thc_shard_range(h->NL, h->NP, rank, nranks, r);
  if (st != THC_OK) return st;
  if (r[1] > r[0] && bad_ptr(B_ov)) return THC_ERR_INVALID_ARG;
  DeviceGuard g(h->device);
  if (!g.ok) return THC_ERR_CUDA;
  st = ensure_workspace(h, h->need_bytes);
  if (st != THC_OK) return st;
  return run_energy(h, static_cast<char*>(h->ws), h->ws_bytes, Xo, Xv, Z, B_ov, nullptr, E_dev, r[1] - r[0]);
}

// ---- second workload ---------------------------------------------------------------------------------
static Need dry_mp2(thc_handle* h) {
  Ctx c{h}; c.dry = true; c.ar.dry = true;
  plan_mp2_density(c, nullptr, nullptr, nullptr, nullptr, nullptr);
  return Need{c.ar.peak, c.splitk_need};
}
static Need dry_als(thc_handle* h, i64 I, i64 J, i64 K, i64 N) {
  Ctx c{h}; c.dry = true; c.ar.dry = true;
  plan_als_update(c, I, J, K, N, nullptr, nullptr, nullptr, nullptr, 1, reinterpret_cast<double*>(static_cast<uintptr_t>(256)));
  return Need{c.ar.peak, c.splitk_need};
}

int64_t thc_workspace_bytes_mp2(const thc_handle* h) {
  return h ? dry_mp2(const_cast<thc_handle*>(h)).total() : (int64_t)THC_ERR_INVALID_ARG;
}

int thc_mp2_density(thc_handle* h, const double* Xo, const double* Xv, const double* Z, double* D_oo, double* D_vv) {
  if (!h || bad_ptr(Xo) || bad_ptr(Xv) || bad_ptr(Z) || bad_ptr(D_oo) || bad_ptr(D_vv)) return THC_ERR_INVALID_ARG;
  DeviceGuard g(h->device);
  if (!g.ok) return THC_ERR_CUDA;
  const Need need = dry_mp2(h);
  int st = ensure_workspace(h, std::max<i64>(h->need_bytes, need.total()));
  if (st != THC_OK) return st;
  Ctx c{h};
  st = make_ctx(c, h, static_cast<char*>(h->ws), h->ws_bytes, need);
  if (st != THC_OK) return st;
  plan_mp2_density(c, Xo, Xv, Z, D_oo, D_vv);
  if (c.ar.overflow) return THC_ERR_NO_MEMORY;
  return c.status;
}

static bool als_dims_ok(int64_t I, int64_t J, int64_t K, int64_t N) {
  const int64_t lim = (int64_t)1 << 31;
  return I > 0 && J > 0 && K > 0 && N > 0 && I < lim && N < lim && J < lim && K < lim && (long double)J * K < (long double)lim &&
         (long double)I * J * K * 8 < 9e18L;
}

int64_t thc_workspace_bytes_als(const thc_handle* h, int64_t I, int64_t J, int64_t K, int64_t N) {
  if (!h || !als_dims_ok(I, J, K, N)) return (int64_t)THC_ERR_INVALID_ARG;
  return dry_als(const_cast<thc_handle*>(h), I, J, K, N).total();
}

int thc_cp_als_update(thc_handle* h, int64_t I, int64_t J, int64_t K, int64_t N, const double* A, const double* Y,
                      const double* Z, double* X, int iters, double* rnorm2) {
  if (!h || !als_dims_ok(I, J, K, N) || iters < 0) return THC_ERR_INVALID_ARG;
  if (bad_ptr(A) || bad_ptr(Y) || bad_ptr(Z) || bad_ptr(X) || (rnorm2 && bad_ptr(rnorm2))) return THC_ERR_INVALID_ARG;
  DeviceGuard g(h->device);
  if (!g.ok) return THC_ERR_CUDA;
  const Need need = dry_als(h, I, J, K, N);
  int st = ensure_workspace(h, std::max<i64>(h->need_bytes, need.total()));
  if (st != THC_OK) return st;
  Ctx c{h};
  st = make_ctx(c, h, static_cast<char*>(h->ws), h->ws_bytes, need);
  if (st != THC_OK) return st;
  plan_als_update(c, I, J, K, N, A, Y, Z, X, iters, rnorm2);
  if (c.ar.overflow) return THC_ERR_NO_MEMORY;
  return c.status;
}

int thc_profile_begin(thc_handle* h, int class_mask) {
  if (!h || class_mask < 0 || class_mask > 7) return THC_ERR_INVALID_ARG;
  h->prof_mask = class_mask;
  h->prof_used = 0;
  return THC_OK;
}

int thc_profile_end(thc_handle* h, double ms[3], int64_t counts[3]) {
  if (!h || !ms || !counts) return THC_ERR_INVALID_ARG;
  DeviceGuard g(h->device);
  if (!g.ok) return THC_ERR_CUDA;
  for (int k = 0; k < 3; k++) { ms[k] = 0.0; counts[k] = 0; h->prof_work[k] = 0.0; }
  cudaError_t e = cudaStreamSynchronize(h->stream);
  if (e != cudaSuccess) { h->last_cuda = (int)e; return THC_ERR_CUDA; }
  h->prof_ms.assign(h->prof_used, 0.f);
  h->prof_done = 0;
  for (size_t k = 0; k < h->prof_used; k++) {
    float t = 0.f;
    e = cudaEventElapsedTime(&t, h->prof_events[2 * k], h->prof_events[2 * k + 1]);
    if (e != cudaSuccess) { h->last_cuda = (int)e; return THC_ERR_CUDA; }
    h->prof_ms[k] = t;
    ms[h->prof_class[k]] += (double)t;
    counts[h->prof_class[k]]++;
    h->prof_work[h->prof_class[k]] += h->prof_flops[k];
  }
  h->prof_done = h->prof_used;
  h->prof_mask = 0;
  h->prof_used = 0;
  return THC_OK;
}

int thc_profile_work(const thc_handle* h, double work[3]) {
  if (!h || !work) return THC_ERR_INVALID_ARG;
  for (int k = 0; k < 3; k++) work[k] = h->prof_work[k];
  return THC_OK;
}

int64_t thc_profile_launches(const thc_handle* h) { return h ? (int64_t)h->prof_done : (int64_t)THC_ERR_INVALID_ARG; }

int thc_profile_launch(const thc_handle* h, int64_t k, int* cls, double* ms, double* work, char* desc, int64_t desc_bytes) {
  if (!h || k < 0 || (size_t)k >= h->prof_done) return THC_ERR_INVALID_ARG;
  if (cls) *cls = h->prof_class[k];
  if (ms) *ms = (double)h->prof_ms[k];
  if (work) *work = h->prof_flops[k];
  if (desc && desc_bytes > 0) {
    strncpy(desc, h->prof_desc[k].c_str(), (size_t)desc_bytes - 1);
    desc[desc_bytes - 1] = 0;
  }
  return THC_OK;
}

int thc_residual_host(thc_handle* h, const double* Xo, const double* Xv, const double* Z, const double* B_ov,
                      const double* B_oo, const void* B_vv, const double* Y, const double* V, const double* eps,
                      double* R_host, double* E_host) {
  if (!h || !R_host) return THC_ERR_INVALID_ARG;
  const double* src[9] = {Xo, Xv, Z, B_ov, B_oo, static_cast<const double*>(B_vv), Y, V, eps};
  for (int k = 0; k < 9; k++) if (bad_ptr(src[k])) return THC_ERR_INVALID_ARG;
  DeviceGuard g(h->device);
  if (!g.ok) return THC_ERR_CUDA;
  const i64 need = need_host(h);
  int st = ensure_workspace(h, need);
  if (st != THC_OK) return st;
  // staging area at the front of the workspace
  i64 sz[9];
  input_doubles(h, sz);
  char* p = reinterpret_cast<char*>((reinterpret_cast<uintptr_t>(h->ws) + 255) / 256 * 256);
  double* dev[9];
  for (int k = 0; k < 9; k++) {
    dev[k] = reinterpret_cast<double*>(p);
    if (sz[k] == 0) { dev[k] = const_cast<double*>(src[k]); continue; }
    cudaError_t e = cudaMemcpyAsync(dev[k], src[k], (size_t)sz[k] * 8, cudaMemcpyHostToDevice, h->stream);
    if (e != cudaSuccess) { h->last_cuda = (int)e; return THC_ERR_CUDA; }
    p += (sz[k] * 8 + 255) / 256 * 256;
  }
  double* Rd = reinterpret_cast<double*>(p);
  p += (h->NP * h->NP * 8 + 255) / 256 * 256;
  const i64 rest = h->ws_bytes - (p - static_cast<char*>(h->ws));
  Inputs in{dev[0], dev[1], dev[2], dev[3], dev[4], dev[5], dev[6], dev[7], dev[8]};
  Outputs out{};
  out.R = Rd;
  if (h->check_symmetry && (st = check_symmetric(h, in, h->NL)) != THC_OK) return st;
  st = run_residual(h, p, rest, in, out);
  if (st != THC_OK) return st;
  cudaError_t e = cudaMemcpyAsync(R_host, Rd, (size_t)h->NP * h->NP * 8, cudaMemcpyDeviceToHost, h->stream);
  if (e != cudaSuccess) { h->last_cuda = (int)e; return THC_ERR_CUDA; }
  if (E_host) {
    st = run_energy(h, p, rest, dev[0], dev[1], dev[2], dev[3], E_host, nullptr);   // synchronises
    if (st != THC_OK) return st;
  }
  e = cudaStreamSynchronize(h->stream);
  if (e != cudaSuccess) { h->last_cuda = (int)e; return THC_ERR_CUDA; }
  return THC_OK;
}

int64_t thc_kernel_launches(const thc_handle* h) { return h ? h->launches : 0; }

// SURVEY.md 8(a) / DESIGN.md section 7: straightforward GEMM order, FMA = 2 flop, no symmetry savings, the G
// intermediates of Alg.6 counted once (re-computation per X-block is not algorithmic work).
double thc_algorithmic_flops(const thc_handle* h) {
  if (!h) return 0.0;
  const double o = (double)h->o, v = (double)h->v, NL = (double)h->NL, NP = (double)h->NP, NX = (double)h->NX;
  const double NP2 = NP * NP, NP3 = NP2 * NP, ov = o * v;
  double f = 0.0;
  f += 2 * (o + v) * NP2 + 2 * NP3;                                                    // H0
  f += NL * (2 * o * o * NP + 2 * o * NP2);                                            // H1
  f += NL * (2 * v * v * NP + 2 * v * NP2);                                            // H2
  f += 5 * NL * NP2;                                                                   // H3
  f += 4 * NL * NP3;                                                                   // H4
  f += NL * (2 * ov * NP + 2 * o * NP2);                                               // H5
  f += NL * (4 * o * NP2 + 2 * ov * NP + 2 * o * o * v + 2 * ov * v);                  // H6
  f += 6 * NP2 * NL;                                                                   // H7
  f += 4 * NP3 + 4 * (o + v) * NP2 + 2 * (o * o + v * v) * NP;                         // H8
  f += 2 * ov * NP2 + 4 * ov * NP2;                                                    // H9 (a),(b): A3, C, D
  f += 2 * ov * NX * NX + NX * (2 * ov * NP + 2 * o * NP2);                            // H9 B_ia^I and G
  f += 2 * (o + v) * NP2 * NX;                                                         // H9 (c): E, F
  f += 5 * NX * NP3;                                                                   // H9 (d): line 11
  f += NP * (2 * o * NP2 + 4 * ov * NP);                                               // H9 (e)
  f += NP * (2 * o * NP2 + 4 * ov * NP);                                               // H10 pass 1
  f += 2 * NP * (4 * o * NX * NX + 4 * ov * NX);                                       // H10 pass 2 (R and S)
  f += 4 * NP2 * ov + 2 * NP * NX * NX + 2 * NP2 * NX;                                 // H10 assembly
  return f;
}

int thc_algorithmic_work(const thc_handle* h, double work[3]) {
  if (!h || !work) return THC_ERR_INVALID_ARG;
  const double NL = (double)h->NL, NP = (double)h->NP, NX = (double)h->NX;
  work[1] = 5 * NX * NP * NP * NP;                      // H9 (d): line 11
  work[2] = 5 * NL * NP * NP;                           // H3
  work[0] = thc_algorithmic_flops(h) - work[1] - work[2];
  return THC_OK;
}

int thc_dgemm(thc_handle* h, int a_kmajor, int b_kmajor, int64_t M, int64_t N, int64_t K, double alpha, const double* A,
              int64_t lda, const double* B, int64_t ldb, double beta, double* C, int64_t ldc) {
  if (!h || bad_ptr(A) || bad_ptr(B) || bad_ptr(C) || M <= 0 || N <= 0 || K <= 0) return THC_ERR_INVALID_ARG;
  const int64_t lim = (int64_t)1 << 31;
  if (M >= lim || N >= lim || K >= lim) return THC_ERR_OVERFLOW;
  if (lda < (a_kmajor ? K : M) || ldb < (b_kmajor ? K : N) || ldc < N) return THC_ERR_INVALID_ARG;
  DeviceGuard g(h->device);
  if (!g.ok) return THC_ERR_CUDA;
  Gemm gm(A, lda, a_kmajor ? 'K' : 'M', B, ldb, b_kmajor ? 'K' : 'N', C, ldc, M, N, K);
  gm.ab(alpha, beta);
  Ctx d{h}; d.dry = true; d.ar.dry = true;
  d.gemm(gm);
  Need need{0, d.splitk_need};
  int st = ensure_workspace(h, std::max<i64>(h->need_bytes, need.total()));
  if (st != THC_OK) return st;
  Ctx c{h};
  st = make_ctx(c, h, static_cast<char*>(h->ws), h->ws_bytes, need);
  if (st != THC_OK) return st;
  c.gemm(gm);
  return c.status;
}

int thc_triple_product(thc_handle* h, int64_t nI, int64_t nPp, int64_t NPp, const double* E, const double* F,
                       const double* G, double* H, int accumulate) {
  if (!h || bad_ptr(E) || bad_ptr(F) || bad_ptr(G) || bad_ptr(H) || nI <= 0 || nPp <= 0 || NPp <= 0) return THC_ERR_INVALID_ARG;
  if (nPp % thc::TP_PT != 0 || NPp % thc::TP_RT != 0) return THC_ERR_INVALID_ARG;
  if (((reinterpret_cast<uintptr_t>(E) | reinterpret_cast<uintptr_t>(F) | reinterpret_cast<uintptr_t>(G) | reinterpret_cast<uintptr_t>(H)) & 15) != 0)
    return THC_ERR_INVALID_ARG;
  DeviceGuard g(h->device);
  if (!g.ok) return THC_ERR_CUDA;
  Ctx c{h};
  c.dry = false;
  c.triple_product(E, F, G, H, nI, nPp, NPp, accumulate);
  return c.status;
}

int thc_probe(thc_handle* h, double out[8]) {
  if (!h || !out) return THC_ERR_INVALID_ARG;
  DeviceGuard g(h->device);
  if (!g.ok) return THC_ERR_CUDA;
  for (int k = 0; k < 8; k++) out[k] = 0.0;
  double* sink = nullptr;
  cudaEvent_t e0, e1;
  if (cudaMalloc(&sink, 64) != cudaSuccess || cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) {
    h->last_cuda = (int)cudaGetLastError();
    return THC_ERR_CUDA;
  }
  int khz = 0;
  cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, h->device);          // maximum SM clock
  const double clk = (double)khz * 1e3;
  const int grid = h->sms, fp_iters = 1 << 16, lds_iters = 1 << 15;
  auto timed = [&](auto launch) -> double {                                 // seconds, best of 3 after a warm-up
    launch();
    float best = 1e30f;
    for (int r = 0; r < 3; r++) {
      cudaEventRecord(e0, h->stream);
      launch();
      cudaEventRecord(e1, h->stream);
      cudaEventSynchronize(e1);
      float ms = 0.f;
      cudaEventElapsedTime(&ms, e0, e1);
      best = std::min(best, ms);
    }
    return (double)best * 1e-3;
  };
  const double warps = (double)grid * thc::PROBE_THREADS / 32, n_fp = (double)fp_iters * thc::PROBE_UNROLL;
  const double dmma_flop = warps * n_fp * 2.0 * 8 * 8 * 4, dfma_flop = warps * 32.0 * n_fp * 2.0;
  out[0] = dmma_flop / timed([&] { thc::probe_fp64_kernel<0><<<grid, thc::PROBE_THREADS, 0, h->stream>>>(sink, fp_iters, 1.25); }) / 1e12;
  out[1] = dfma_flop / timed([&] { thc::probe_fp64_kernel<1><<<grid, thc::PROBE_THREADS, 0, h->stream>>>(sink, fp_iters, 1.25); }) / 1e12;
  out[2] = (dmma_flop + dfma_flop) / timed([&] { thc::probe_fp64_kernel<2><<<grid, thc::PROBE_THREADS, 0, h->stream>>>(sink, fp_iters, 1.25); }) / 1e12;
  unsigned* usink = reinterpret_cast<unsigned*>(sink);
  const double lanes_loads = (double)grid * thc::PROBE_THREADS * lds_iters * 8.0;
  out[3] = lanes_loads * 4 / timed([&] { thc::probe_lds_kernel<4><<<grid, thc::PROBE_THREADS, 0, h->stream>>>(usink, lds_iters, 0u); }) / clk / grid;
  out[4] = lanes_loads * 8 / timed([&] { thc::probe_lds_kernel<8><<<grid, thc::PROBE_THREADS, 0, h->stream>>>(usink, lds_iters, 0u); }) / clk / grid;
  out[5] = lanes_loads * 16 / timed([&] { thc::probe_lds_kernel<16><<<grid, thc::PROBE_THREADS, 0, h->stream>>>(usink, lds_iters, 0u); }) / clk / grid;
  out[6] = clk / 1e6;
  h->launches += 24;
  cudaError_t e = cudaGetLastError();
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(sink);
  if (e != cudaSuccess) { h->last_cuda = (int)e; return THC_ERR_CUDA; }
  return THC_OK;
}

const char* thc_strerror(int status) {
  switch (status) {
    case THC_OK: return "ok";
    case THC_ERR_INVALID_ARG: return "invalid argument (null or misaligned pointer, bad size)";
    case THC_ERR_OVERFLOW: return "size overflow";
    case THC_ERR_NO_MEMORY: return "workspace too small or device allocation failed";
    case THC_ERR_CUDA: return "CUDA error (see thc_last_error)";
    case THC_ERR_NO_DEVICE: return "no sm_100 CUDA device";
    case THC_ERR_PROVIDER: return "B_vv provider callback failed";
    case THC_ERR_STATIC_LIMIT: return "thc_dgemm_static: splits * M * N * 8 bytes exceed THC_STATIC_SCRATCH_BYTES";
    default: return "unknown status";
  }
}

int thc_last_error(const thc_handle* h) { return h ? h->last_cuda : 0; }
int thc_last_cuda_error(const thc_handle* h) { return thc_last_error(h); }

}  // extern "C"

// ---- allocation-free split-K DGEMM (include/thc.h: thc_static_init, thc_dgemm_static) -----------------------------------
// The split-K partial tiles live in a static device array: one per GPU per process, from library load until exit.
// In host code `thc_static_scratch` is only a host-side stand-in for the symbol, never a device address: the address
// that the kernels get comes from cudaGetSymbolAddress, asked once per device with that device current.
static __device__ __align__(256) double thc_static_scratch[THC_STATIC_SCRATCH_BYTES / 8];

namespace {
constexpr int STATIC_MAX_DEVICES = 64;
struct StaticDev { bool ready = false; double* scratch = nullptr; int sms = 0; };
StaticDev g_static_dev[STATIC_MAX_DEVICES];
std::mutex g_static_mutex;

// set-up of the current device (the caller holds a DeviceGuard on `device`)
int static_init_current(int device) {
  std::lock_guard<std::mutex> lock(g_static_mutex);
  StaticDev& d = g_static_dev[device];
  if (d.ready) return THC_OK;
  int major = 0;
  if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, device) != cudaSuccess || major != 10) {
    cudaGetLastError();
    return THC_ERR_NO_DEVICE;
  }
  double* ptr = nullptr;
  if (cudaGetSymbolAddress(reinterpret_cast<void**>(&ptr), thc_static_scratch) != cudaSuccess || !ptr) { cudaGetLastError(); return THC_ERR_CUDA; }
  if (cudaDeviceGetAttribute(&d.sms, cudaDevAttrMultiProcessorCount, device) != cudaSuccess || d.sms <= 0) { cudaGetLastError(); return THC_ERR_CUDA; }
  const int sm = thc::gemm_smem_bytes(64, 64, 16, 4, true, true);        // 64 KB: above the 48 KB default
  if (cudaFuncSetAttribute(thc::dgemm_kernel<THC_SMALL, true, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm) != cudaSuccess ||
      cudaFuncSetAttribute(thc::dgemm_kernel<THC_SMALL, true, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm) != cudaSuccess) {
    cudaGetLastError();
    return THC_ERR_CUDA;
  }
  d.scratch = ptr;
  d.ready = true;
  return THC_OK;
}
}  // namespace

int thc_static_init(int device) {
  if (device < 0 && cudaGetDevice(&device) != cudaSuccess) { cudaGetLastError(); return THC_ERR_NO_DEVICE; }
  if (device >= STATIC_MAX_DEVICES) return THC_ERR_INVALID_ARG;
  DeviceGuard g(device);
  if (!g.ok) return THC_ERR_CUDA;
  return static_init_current(device);
}

int thc_dgemm_static(int device, void* stream, int64_t M, int64_t N, int64_t K, int splits, double alpha, const double* A,
                     int64_t lda, const double* B, int64_t ldb, double beta, double* C, int64_t ldc) {
  if (bad_ptr(A) || bad_ptr(B) || bad_ptr(C) || M <= 0 || N <= 0 || K <= 0 || splits < 0) return THC_ERR_INVALID_ARG;
  const int64_t lim = (int64_t)1 << 31;
  if (M >= lim || N >= lim || K >= lim) return THC_ERR_OVERFLOW;
  if (lda < K || ldb < K || ldc < N) return THC_ERR_INVALID_ARG;
  const i64 per = M * N, cap = THC_STATIC_SCRATCH_BYTES / 8;
  if (splits > 1 && (splits > cap || per > cap / splits)) return THC_ERR_STATIC_LIMIT;
  if (device < 0 && cudaGetDevice(&device) != cudaSuccess) { cudaGetLastError(); return THC_ERR_NO_DEVICE; }
  if (device >= STATIC_MAX_DEVICES) return THC_ERR_INVALID_ARG;
  DeviceGuard g(device);
  if (!g.ok) return THC_ERR_CUDA;
  int st = static_init_current(device);
  if (st != THC_OK) return st;
  const StaticDev& d = g_static_dev[device];
  const i64 tiles = ((M + 63) / 64) * ((N + 63) / 64), kiters = (K + 15) / 16;
  if (tiles >= lim) return THC_ERR_OVERFLOW;
  if (splits == 0) {
    // about two waves of three 64 x 64 CTAs per SM, at least four k-tiles per split, within the scratch
    const i64 want = std::max<i64>(1, (i64)d.sms * 6 / tiles);
    splits = (int)std::max<i64>(1, std::min<i64>(std::min<i64>(want, kiters / 4), std::min<i64>(cap / per, 64)));
  }
  splits = (int)std::min<i64>(splits, kiters);              // no empty K ranges
  if (splits > 65535) return THC_ERR_INVALID_ARG;           // grid.z
  cudaStream_t s = static_cast<cudaStream_t>(stream);

  thc::GemmParams p{};
  p.A = A; p.B = B; p.aux = nullptr;
  p.M = (int)M; p.N = (int)N; p.K = (int)K;
  p.lda = lda; p.ldb = ldb;
  p.batch = 1; p.kbatch = 1; p.splits = splits;
  p.alpha = alpha; p.beta = beta;
  if (splits > 1) { p.C = d.scratch; p.ldc = N; p.sCb = per; p.sCs = per; }
  else            { p.C = C; p.ldc = ldc; }
  const bool al16 = ((reinterpret_cast<uintptr_t>(A) | reinterpret_cast<uintptr_t>(B)) & 15) == 0 && (lda & 1) == 0 && (ldb & 1) == 0;
  const int sm = thc::gemm_smem_bytes(64, 64, 16, 4, true, true);
  const dim3 grid((unsigned)tiles, 1, (unsigned)splits);
  if (al16) thc::dgemm_kernel<THC_SMALL, true, true, true><<<grid, thc::SMALL_THREADS, sm, s>>>(p);
  else      thc::dgemm_kernel<THC_SMALL, true, true, false><<<grid, thc::SMALL_THREADS, sm, s>>>(p);
  if (cudaPeekAtLastError() != cudaSuccess) { cudaGetLastError(); return THC_ERR_CUDA; }
  if (splits > 1) {
    thc::ReduceParams r{};
    r.part = d.scratch; r.dst = C; r.aux = nullptr;
    r.M = (int)M; r.N = (int)N; r.batch = 1; r.splits = splits;
    r.ldd = ldc; r.alpha = alpha; r.beta = beta;
    const int blocks = (int)std::max<i64>(1, std::min<i64>((per + 255) / 256, (i64)d.sms * 16));
    thc::reduce_splits_kernel<<<blocks, 256, 0, s>>>(r);
    if (cudaPeekAtLastError() != cudaSuccess) { cudaGetLastError(); return THC_ERR_CUDA; }
  }
  return THC_OK;
}
