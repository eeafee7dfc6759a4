// Hadamard / reduction kernels (HBM-streaming) and the Alg.6 line-11 triple-product kernel (FP64 FMA pipe).
// Citations are PAPER.md line numbers.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "thc_gemm.cuh"

namespace thc {

typedef long long i64;

#define THC_GRID_STRIDE(idx, total) \
  for (i64 idx = (i64)blockIdx.x * blockDim.x + threadIdx.x; idx < (total); idx += (i64)gridDim.x * blockDim.x)

// out[c][r] = in[r][c]   (small factor matrices only)
__global__ void transpose_kernel(const double* __restrict__ in, double* __restrict__ out, int rows, int cols) {
  __shared__ double tile[32][33];
  int c0 = blockIdx.x * 32, r0 = blockIdx.y * 32;
  for (int j = threadIdx.y; j < 32; j += blockDim.y) {
    int r = r0 + j, c = c0 + threadIdx.x;
    if (r < rows && c < cols) tile[j][threadIdx.x] = in[(i64)r * cols + c];
  }
  __syncthreads();
  for (int j = threadIdx.y; j < 32; j += blockDim.y) {
    int c = c0 + j, r = r0 + threadIdx.x;
    if (r < rows && c < cols) out[(i64)c * rows + r] = tile[threadIdx.x][j];
  }
}

__global__ void fill_kernel(double* __restrict__ x, i64 n, double val) {
  THC_GRID_STRIDE(i, n) x[i] = val;
}

// out = a .* b                                   (w = o .* v, Alg.3 l.596, Alg.7 l.736, Alg.9 l.817)
__global__ void hadamard_kernel(const double* a, const double* b, double* out, i64 n) {      // out may alias a or b
  THC_GRID_STRIDE(i, n) out[i] = a[i] * b[i];
}

// out = ca * a + cb * b
__global__ void axpby_kernel(const double* a, const double* b, double ca, double cb, double* out, i64 n) {   // out may alias a or b
  THC_GRID_STRIDE(i, n) out[i] = ca * a[i] + cb * b[i];
}

// out = a .* b - c .* d                          (E = o .* v~ - o~ .* v, Alg.9 line 9 l.835)
__global__ void had2_diff_kernel(const double* __restrict__ a, const double* __restrict__ b, const double* __restrict__ c,
                                 const double* __restrict__ d, double* __restrict__ out, i64 n) {
  THC_GRID_STRIDE(i, n) out[i] = a[i] * b[i] - c[i] * d[i];
}

// Alg.1 lines 8, 12, 13 (l.502-518) and Alg.3 line 7 (l.587), for nl Cholesky vectors at once:
//   C^l = v .* Mo^l - o .* Mv^l   (written over Mo),   C3 += sum_l Mo^l .* Mv^l
__global__ void combine_kernel(double* __restrict__ Mo, const double* __restrict__ Mv, const double* __restrict__ omat,
                               const double* __restrict__ vmat, double* __restrict__ C3, i64 np2, int nl) {
  THC_GRID_STRIDE(i, np2) {
    double ov = omat[i], vv = vmat[i], c3 = 0.0;
    for (int l = 0; l < nl; l++) {
      double mo = Mo[(i64)l * np2 + i], mv = Mv[(i64)l * np2 + i];
      c3 = fma(mo, mv, c3);
      Mo[(i64)l * np2 + i] = vv * mo - ov * mv;
    }
    C3[i] += c3;
  }
}

// FvoT[i][a] = (eps[o+a] - eps[i]) * t1[i][a]: the one-electron part of the dressed Fock matrix F^_ai (canonical orbitals)
__global__ void t1_eps_kernel(const double* __restrict__ eps, const double* __restrict__ t1, double* __restrict__ out, int o, int v) {
  THC_GRID_STRIDE(idx, (i64)o * v) {
    const int i = (int)(idx / v), a = (int)(idx % v);
    out[idx] = (eps[o + a] - eps[i]) * t1[idx];
  }
}

// Alg.4 / Alg.5 line 13 (l.640, l.677): sigma^{XX'} += sum_pairs J_pair^{XX'} fa_pair[X] fb_pair[X'] for the n1 x n2 pairs
// (i1, i2) of a block; J is [(i1, i2)][n][n], fa = FA[i1][.], fb = FB[i2][.] (A^{XX'} = y^X y^{X'} of line 3).
__global__ void pair_accumulate_kernel(const double* __restrict__ J, const double* __restrict__ FA, i64 ldfa,
                                       const double* __restrict__ FB, i64 ldfb, double* __restrict__ out, int n, int n1, int n2) {
  const i64 nn = (i64)n * n;
  THC_GRID_STRIDE(idx, nn) {
    const int X = (int)(idx / n), Xp = (int)(idx % n);
    double s = 0.0;
    for (int i1 = 0; i1 < n1; i1++) {
      const double fa = FA[(i64)i1 * ldfa + X];
      double s1 = 0.0;
      for (int i2 = 0; i2 < n2; i2++) s1 = fma(J[((i64)i1 * n2 + i2) * nn + idx], FB[(i64)i2 * ldfb + Xp], s1);
      s = fma(fa, s1, s);
    }
    out[idx] += s;
  }
}

// d[P] = A[P][P]
__global__ void diag_kernel(const double* __restrict__ A, double* __restrict__ d, int n) {
  THC_GRID_STRIDE(idx, (i64)n) d[idx] = A[idx * n + idx];
}

// ---- preconditioned conjugate gradients on S x_i = R_i, one system per row i (App.I l.373: "solved on the GPU by
// the preconditioned conjugate gradient method using the diagonal of S as the preconditioner"; the rows are independent).
// One warp per row, lane j takes columns j, j + 32, ...; xor-shuffle reductions (fixed order: deterministic).
__device__ __forceinline__ double warp_sum_all(double s) {
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
  return s;
}
// start: z = r / d, p = z, rz[i] = r_i . z_i      (r = R - X S was formed by a GEMM)
__global__ void pcg_init_kernel(const double* __restrict__ r, const double* __restrict__ d, double* __restrict__ p,
                                double* __restrict__ rz, int nrows, int n) {
  const int lane = threadIdx.x & 31;
  for (i64 row = ((i64)blockIdx.x * blockDim.x + threadIdx.x) >> 5; row < nrows; row += ((i64)gridDim.x * blockDim.x) >> 5) {
    const double* rr = r + row * n;
    double* pp = p + row * n;
    double s = 0.0;
    for (int c = lane; c < n; c += 32) {
      const double z = rr[c] / d[c];
      pp[c] = z;
      s += rr[c] * z;
    }
    s = warp_sum_all(s);
    if (lane == 0) rz[row] = s;
  }
}
// one iteration given Sp = S p:  alpha = rz / p.Sp,  x += alpha p,  r -= alpha Sp,  z = r / d,  beta = r.z / rz,  p = z + beta p.
// A row with p.Sp = 0 takes a zero step, a row with rz = 0 keeps beta = 0 (exactly converged rows stay put; oracle/als.py).
__global__ void pcg_iter_kernel(double* __restrict__ x, double* __restrict__ r, double* __restrict__ p, const double* __restrict__ Sp,
                                const double* __restrict__ d, double* __restrict__ rz, int nrows, int n) {
  const int lane = threadIdx.x & 31;
  for (i64 row = ((i64)blockIdx.x * blockDim.x + threadIdx.x) >> 5; row < nrows; row += ((i64)gridDim.x * blockDim.x) >> 5) {
    double* xx = x + row * n;
    double* rr = r + row * n;
    double* pp = p + row * n;
    const double* sp = Sp + row * n;
    double pSp = 0.0;
    for (int c = lane; c < n; c += 32) pSp += pp[c] * sp[c];
    pSp = warp_sum_all(pSp);
    const double rz_old = rz[row];
    const double alpha = pSp != 0.0 ? rz_old / pSp : 0.0;
    double rz_new = 0.0;
    for (int c = lane; c < n; c += 32) {
      xx[c] += alpha * pp[c];
      const double rc = rr[c] - alpha * sp[c];
      rr[c] = rc;
      rz_new += rc * (rc / d[c]);
    }
    rz_new = warp_sum_all(rz_new);
    const double beta = rz_old != 0.0 ? rz_new / rz_old : 0.0;
    for (int c = lane; c < n; c += 32) pp[c] = rr[c] / d[c] + beta * pp[c];
    __syncwarp();
    if (lane == 0) rz[row] = rz_new;
  }
}

// out[b*ldo + r] = sum_{i<n} X[r*ldx + i] * T[b*sTb + r*ldT + i]      (a^L_P: Alg.2 l.541, Alg.8 l.788; C7: Alg.7 line 9 l.749)
// Eight lanes share a row (lane j takes i = j, j + 8, ...: 64-byte coalesced segments), xor-shuffle reduction.
__global__ void rowdot_kernel(const double* __restrict__ X, i64 ldx, const double* __restrict__ T, i64 sTb, i64 ldT,
                              double* __restrict__ out, i64 ldo, int nb, int nr, int n) {
  const i64 total = (i64)nb * nr;
  const int sub = threadIdx.x & 7;
  const i64 rows_per_pass = (i64)gridDim.x * (blockDim.x >> 3);
  const i64 passes = (total + rows_per_pass - 1) / rows_per_pass;      // every lane runs every pass (full-warp shuffles)
  i64 idx = (i64)blockIdx.x * (blockDim.x >> 3) + (threadIdx.x >> 3);
  for (i64 it = 0; it < passes; it++, idx += rows_per_pass) {
    double s = 0.0;
    const bool ok = idx < total;
    int r = 0, b = 0;
    if (ok) {
      r = (int)(idx % nr); b = (int)(idx / nr);
      const double* x = X + (i64)r * ldx;
      const double* tt = T + (i64)b * sTb + (i64)r * ldT;
      for (int i = sub; i < n; i += 8) s = fma(x[i], tt[i], s);
    }
    s += __shfl_xor_sync(0xffffffffu, s, 1);
    s += __shfl_xor_sync(0xffffffffu, s, 2);
    s += __shfl_xor_sync(0xffffffffu, s, 4);
    if (ok && sub == 0) out[(i64)b * ldo + r] = s;
  }
}

// out[b*ldo + c] = sum_{i<n} X[i*ldx + c] * T[b*sTb + i*ldT + c]      (d^L_P: Alg.2 l.549,557; sigma6 row: Alg.6 line 15 l.724)
__global__ void coldot_kernel(const double* __restrict__ X, i64 ldx, const double* __restrict__ T, i64 sTb, i64 ldT,
                              double* __restrict__ out, i64 ldo, int nb, int nc, int n) {
  i64 total = (i64)nb * nc;
  THC_GRID_STRIDE(idx, total) {
    int c = (int)(idx % nc), b = (int)(idx / nc);
    const double* tt = T + (i64)b * sTb + c;
    double s = 0.0;
    for (int i = 0; i < n; i++) s = fma(X[(i64)i * ldx + c], tt[(i64)i * ldT], s);
    out[(i64)b * ldo + c] = s;
  }
}

// out[(b,i)][c] = alpha * X[i][c] * Mrow[b][c] (+ add[(b,i)][c])       b < nb, i < n, c < nc
// (Xo .* v_P, Alg.7 line 6 l.743 in scaled-factor form; 2 Xo .* K_P, Alg.7 line 4 l.739; Z_Q .* Xo, Alg.6 line 1 l.683;
//  V_I .* Yo, Alg.6 line 2 l.686)
__global__ void rowscale_kernel(const double* __restrict__ X, i64 ldx, const double* __restrict__ Mrow, i64 ldm,
                                const double* __restrict__ add, double alpha, double* __restrict__ out, int nb, int n, int nc) {
  i64 total = (i64)nb * n * nc;
  THC_GRID_STRIDE(idx, total) {
    int c = (int)(idx % nc);
    i64 r = idx / nc;
    int i = (int)(r % n), b = (int)(r / n);
    double val = alpha * X[(i64)i * ldx + c] * Mrow[(i64)b * ldm + c];
    if (add) val += add[idx];
    out[idx] = val;
  }
}

// the same, two columns per thread with 16-byte accesses (nc, ldx, ldm even; all pointers 16-byte aligned)
__global__ void rowscale2_kernel(const double* __restrict__ X, i64 ldx, const double* __restrict__ Mrow, i64 ldm,
                                 const double* __restrict__ add, double alpha, double* __restrict__ out, int nb, int n, int nc) {
  const int nc2 = nc >> 1;
  const i64 total = (i64)nb * n * nc2;
  THC_GRID_STRIDE(idx, total) {
    const int c = (int)(idx % nc2) * 2;
    const i64 r = idx / nc2;
    const int i = (int)(r % n), b = (int)(r / n);
    const double2 x = *reinterpret_cast<const double2*>(X + (i64)i * ldx + c);
    const double2 m = *reinterpret_cast<const double2*>(Mrow + (i64)b * ldm + c);
    double2 val = make_double2(alpha * x.x * m.x, alpha * x.y * m.y);
    if (add) { const double2 a = *reinterpret_cast<const double2*>(add + 2 * idx); val.x += a.x; val.y += a.y; }
    *reinterpret_cast<double2*>(out + 2 * idx) = val;
  }
}

// T[(b,i)][c] = alpha * T[(b,i)][c] * Mrow[b][c]   in place            (-(SZ) .* o_P, Alg.7 line 6/7 l.743-745)
__global__ void rowscale_inplace_kernel(double* __restrict__ T, const double* __restrict__ Mrow, i64 ldm, double alpha,
                                        int nb, int n, int nc) {
  i64 total = (i64)nb * n * nc;
  THC_GRID_STRIDE(idx, total) {
    int c = (int)(idx % nc);
    int b = (int)((idx / nc) / n);
    T[idx] = alpha * T[idx] * Mrow[(i64)b * ldm + c];
  }
}

// Qm[i][(l,P)] = 2 Xo[i][P] * ZA[l][P] - G1[i][(l,P)]   in place on G1   (Alg.8 line 7 l.792 folded into line 8)
__global__ void qm_kernel(double* __restrict__ G1, const double* __restrict__ Xo, const double* __restrict__ ZA, int o, int nl, int NP) {
  i64 total = (i64)o * nl * NP;
  THC_GRID_STRIDE(idx, total) {
    int P = (int)(idx % NP);
    i64 r = idx / NP;
    int l = (int)(r % nl), i = (int)(r / nl);
    G1[idx] = 2.0 * Xo[(i64)i * NP + P] * ZA[(i64)l * NP + P] - G1[idx];
  }
}

// out = scale * (P + P^T)                        (Alg.3 line 12 l.601; Alg.9 line 10 l.839)
__global__ void symmetrize_kernel(const double* __restrict__ Pm, double* __restrict__ out, int n, double scale) {
  __shared__ double tile[32][33];
  int bx = blockIdx.x, by = blockIdx.y;
  for (int j = threadIdx.y; j < 32; j += blockDim.y) {
    int r = bx * 32 + j, c = by * 32 + threadIdx.x;   // element of the transposed tile
    if (r < n && c < n) tile[j][threadIdx.x] = Pm[(i64)r * n + c];
  }
  __syncthreads();
  for (int j = threadIdx.y; j < 32; j += blockDim.y) {
    int r = by * 32 + j, c = bx * 32 + threadIdx.x;
    if (r < n && c < n) out[(i64)r * n + c] = scale * (Pm[(i64)r * n + c] + tile[threadIdx.x][j]);
  }
}

// A[m][n] = A[n][m] for m > n   (completes a symmetric matrix whose GEMM computed the upper triangle only)
__global__ void mirror_upper_kernel(double* __restrict__ A, int n) {
  __shared__ double tile[32][33];
  A += (i64)blockIdx.z * n * n;                        // grid.z = batch of densely packed n x n matrices
  const int bx = blockIdx.x, by = blockIdx.y;          // source tile (rows by, cols bx) with by <= bx
  if (by > bx) return;
  for (int j = threadIdx.y; j < 32; j += blockDim.y) {
    int r = by * 32 + j, c = bx * 32 + threadIdx.x;
    if (r < n && c < n) tile[j][threadIdx.x] = A[(i64)r * n + c];
  }
  __syncthreads();
  for (int j = threadIdx.y; j < 32; j += blockDim.y) {
    int r = bx * 32 + j, c = by * 32 + threadIdx.x;    // destination element (r, c) = source (c, r)
    if (r < n && c < n && r > c) A[(i64)r * n + c] = tile[threadIdx.x][j];
  }
}

// FooT[i][j] = delta_ij eps[i] + xi_oo[j][i];  Fvv[a][b] = delta_ab eps[o+a] + xi_vv[a][b]   (Alg.9 lines 5-6 l.823-827)
__global__ void fock_kernel(const double* __restrict__ eps, const double* __restrict__ xi_oo, const double* __restrict__ xi_vv,
                            double* __restrict__ FooT, double* __restrict__ Fvv, int o, int v) {
  i64 total = (i64)o * o + (i64)v * v;
  THC_GRID_STRIDE(idx, total) {
    if (idx < (i64)o * o) {
      int i = (int)(idx / o), j = (int)(idx % o);
      FooT[idx] = xi_oo[(i64)j * o + i] + (i == j ? eps[i] : 0.0);
    } else {
      i64 k = idx - (i64)o * o;
      int a = (int)(k / v), b = (int)(k % v);
      Fvv[k] = xi_vv[k] + (a == b ? eps[o + a] : 0.0);
    }
  }
}

// thc_options.check_symmetry: out[0] = max |A_b[i][j] - A_b[j][i]|, out[1] = max |A_b[i][j]| over nbatch densely packed
// n x n matrices, as the bit patterns of non-negative doubles (which order like unsigned integers).
__global__ void asym_max_kernel(const double* __restrict__ A, int n, i64 nbatch, unsigned long long* __restrict__ out) {
  const i64 total = nbatch * n * n;
  double d = 0.0, m = 0.0;
  THC_GRID_STRIDE(idx, total) {
    const int j = (int)(idx % n);
    const i64 r = idx / n;
    const int i = (int)(r % n);
    const double x = A[idx];
    m = fmax(m, fabs(x));
    if (j > i) d = fmax(d, fabs(x - A[(r - i + j) * n + i]));
  }
  for (int off = 16; off > 0; off >>= 1) {
    d = fmax(d, __shfl_xor_sync(0xffffffffu, d, off));
    m = fmax(m, __shfl_xor_sync(0xffffffffu, m, off));
  }
  if ((threadIdx.x & 31) == 0) {
    atomicMax(out, (unsigned long long)__double_as_longlong(d));
    atomicMax(out + 1, (unsigned long long)__double_as_longlong(m));
  }
}

// R = sum of up to six terms
__global__ void sum6_kernel(const double* a, const double* b, const double* c, const double* d, const double* e,
                            const double* f, double* __restrict__ out, i64 n) {
  THC_GRID_STRIDE(i, n) {
    double s = 0.0;
    if (a) s += a[i];
    if (b) s += b[i];
    if (c) s += c[i];
    if (d) s += d[i];
    if (e) s += e[i];
    if (f) s += f[i];
    out[i] = s;
  }
}

// ---- energy reductions (H12): block partial sums in double-double-free pairwise form, final sum on one block.
__device__ __forceinline__ double block_sum(double v) {
  __shared__ double sh[32];
  for (int off = 16; off > 0; off >>= 1) v += __shfl_down_sync(0xffffffffu, v, off);
  int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  __syncthreads();
  if (l == 0) sh[w] = v;
  __syncthreads();
  int nw = (blockDim.x + 31) >> 5;
  v = (threadIdx.x < nw) ? sh[threadIdx.x] : 0.0;
  if (w == 0)
    for (int off = 16; off > 0; off >>= 1) v += __shfl_down_sync(0xffffffffu, v, off);
  return v;   // valid on thread 0
}

// partial[blockIdx.x] = sum_i a[i] * b[i] over this block's grid-stride share
__global__ void dot_partial_kernel(const double* __restrict__ a, const double* __restrict__ b, i64 n, double* __restrict__ partial) {
  double s = 0.0;
  THC_GRID_STRIDE(i, n) s = fma(a[i], b[i], s);
  s = block_sum(s);
  if (threadIdx.x == 0) partial[blockIdx.x] = s;
}

// partial[block] = sum over the 32x32 tile pair {(bx,by), (by,bx)} of Z[P][Q] * E[l][P][Q] * E[l][Q][P].  Z is symmetric
// (thc.h), so the two tiles of a pair contribute the same amount: only blocks with bx <= by work (each reads both
// tiles once -- E is streamed exactly once overall) and off-diagonal pairs count twice; blocks with bx > by write 0.
// grid = (tiles, tiles, nl), block (32, 8).
__global__ void zee_partial_kernel(const double* __restrict__ Z, const double* __restrict__ E, int NP, double* __restrict__ partial) {
  __shared__ double tile[32][33];
  __shared__ double sh[8];
  const int bx = blockIdx.x, by = blockIdx.y;
  const i64 slot = ((i64)blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x;
  if (bx > by) {
    if (threadIdx.x == 0 && threadIdx.y == 0) partial[slot] = 0.0;
    return;
  }
  const double* El = E + (i64)blockIdx.z * NP * NP;
  for (int j = threadIdx.y; j < 32; j += blockDim.y) {
    int r = bx * 32 + j, c = by * 32 + threadIdx.x;
    tile[j][threadIdx.x] = (r < NP && c < NP) ? El[(i64)r * NP + c] : 0.0;
  }
  __syncthreads();
  double s = 0.0;
  for (int j = threadIdx.y; j < 32; j += blockDim.y) {
    int r = by * 32 + j, c = bx * 32 + threadIdx.x;
    if (r < NP && c < NP) s = fma(Z[(i64)r * NP + c] * El[(i64)r * NP + c], tile[threadIdx.x][j], s);
  }
  if (bx != by) s *= 2.0;
  for (int off = 16; off > 0; off >>= 1) s += __shfl_down_sync(0xffffffffu, s, off);
  if (threadIdx.x == 0) sh[threadIdx.y] = s;
  __syncthreads();
  if (threadIdx.x == 0 && threadIdx.y == 0) {
    double tot = 0.0;
    for (int k = 0; k < (int)blockDim.y; k++) tot += sh[k];
    partial[slot] = tot;
  }
}

// out[0] = ca * sum(pa[0..na)) + cb * sum(pb[0..nb))     (one block; Kahan-compensated per thread, then tree)
__global__ void final_sum_kernel(const double* __restrict__ pa, i64 na, double ca, const double* __restrict__ pb, i64 nb,
                                 double cb, double* __restrict__ out, int accumulate) {
  double s = 0.0, comp = 0.0;
  for (i64 i = threadIdx.x; i < na + nb; i += blockDim.x) {
    double x = (i < na) ? ca * pa[i] : cb * pb[i - na];
    double y = x - comp, tt = s + y;
    comp = (tt - s) - y;
    s = tt;
  }
  s = block_sum(s);
  if (threadIdx.x == 0) out[0] = accumulate ? out[0] + s : s;
}

}  // namespace thc
