/* thc.h -- C ABI of the B200 (sm_100a) THC-RR-CCSD projected doubles residual library.
 *
 * What it computes (arXiv 2111.11473, "Rank-reduced coupled-cluster III"; line numbers are PAPER.md's):
 *
 *   R_PQ = sum_ijab Xo[i,P] Xv[a,P] Omega_ijab Xo[j,Q] Xv[b,Q]            (Eq.6 l.82, Eq.23 l.193)
 *
 * with the doubles amplitudes held only as THC factors t_ij^ab = sum_PQ Xo_iP Xv_aP Z_PQ Xo_jQ Xv_bQ
 * (Eq.23 l.193), the ERIs as Cholesky vectors B^L_pq (Eq.24 l.199, t1 = 0) and, for the T2^2 terms, as THC
 * grid factors <ia|jb> = sum_IJ Yo_iI Yv_aI V_IJ Yo_jJ Yv_bJ (Eq.17 l.141).  Omega is the closed-shell CCSD
 * doubles residual evaluated term by term with the paper's factorised algorithms:
 *
 *   term 0  sigma1  Alg.1 (l.480-530)  Eq.28       term 3  sigma6  Alg.6 (l.682-730)  Eqs.32+33 = Eq.34
 *   term 1  sigma2  Alg.2 (l.532-567)  Eq.29       term 4  sigma7  Alg.7 (l.732-773)  Eqs.35-37 (prefactor 1/2)
 *   term 2  sigma3  Alg.3 (l.569-606)  Eq.31       term 5  sigma9  Alg.9 (l.811-843)  Eq.41, xi from Alg.8 l.5-10
 *
 * and E = sum_ijab (2 t_ij^ab - t_ij^ba)(ia|jb) (l.80; Cholesky ERIs).  Readings of garbled passages: DESIGN.md.
 *
 * Conventions
 *   - All arrays are FP64, row-major, last index contiguous:
 *       Xo[o][NP]  Xv[v][NP]  Z[NP][NP] (symmetric)  B_oo[NL][o][o]  B_ov[NL][o][v]  B_vv[NL][v][v] (each
 *       B^L symmetric)  Y[o+v][NX] (occupied rows first)  V[NX][NX] (symmetric)  eps[o+v] (occupied first)
 *       R[NP][NP].
 *   - Z, V and every B^L are ASSUMED symmetric and the library relies on it: symmetric products (sigma1, the
 *     half-transforms M^{o,L}, M^{v,L}, the energy reduction) are evaluated on the upper triangle and mirrored.  The
 *     hot path does not check; thc_options.check_symmetry turns on a debug pass that does.
 *   - "device pointer" = memory of the handle's CUDA device; "host pointer" = ordinary host memory (pinned
 *     memory makes the copies asynchronous but is not required).
 *   - The caller owns every input and output buffer; inputs are never modified.  The library owns only the
 *     handle.  Scratch memory is a single workspace that the caller may provide (thc_set_workspace, e.g. a
 *     torch allocation) or that the library allocates itself with cudaMalloc on first use.
 *   - Device entry points enqueue work on the handle's stream (thc_set_stream; default stream 0) and return
 *     without synchronising; outputs are valid after the stream has been synchronised.
 *   - Every function returns THC_OK (0) or a negative thc_status; nothing throws or aborts.  The failing CUDA
 *     error (if any) is kept in the handle: thc_last_error.
 *   - Pointers must be 8-byte aligned; 16-byte alignment (and even o, v, NP, NX) selects the vectorised
 *     load path, anything else the scalar one.  There is no CPU fallback of any kind.
 *   - The long launches of Alg.6 line 11 are cooperative launches (one CTA per SM, the CTAs wait for one another at
 *     intervals so that they share operand tiles in L2): they start once every SM is free, so work of other streams
 *     that occupies SMs delays them.
 */
#ifndef THC_H_
#define THC_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct thc_handle thc_handle;

typedef enum {
  THC_OK = 0,
  THC_ERR_INVALID_ARG = -1,   /* null pointer, non-positive size, misaligned pointer            */
  THC_ERR_OVERFLOW = -2,      /* a buffer size does not fit in 63 bits                          */
  THC_ERR_NO_MEMORY = -3,     /* workspace too small / cudaMalloc failed                        */
  THC_ERR_CUDA = -4,          /* a CUDA call or kernel launch failed (see thc_last_error)       */
  THC_ERR_NO_DEVICE = -5,     /* no sm_100 device visible                                       */
  THC_ERR_PROVIDER = -6,      /* a thc_bvv_provider callback returned non-zero                   */
  THC_ERR_STATIC_LIMIT = -7   /* thc_dgemm_static: needs more than THC_STATIC_SCRATCH_BYTES     */
} thc_status;

/* Where the vv Cholesky blocks B_vv[NL][v][v] live (PAPER.md l.191-195 keeps the 3-index arrays off the GPU and
 * streams them; at the paper-scale config B_vv is ~304 GB and can never be resident):
 *   THC_BVV_DEVICE    B_vv is a device pointer to the whole array (default).
 *   THC_BVV_HOST      B_vv is a HOST pointer to the whole array (pinned memory makes the copies overlap); the library
 *                     copies one L-block at a time into a double buffer on its own copy stream, overlapped with the
 *                     GEMMs of the previous block.
 *   THC_BVV_PROVIDER  B_vv points to a thc_bvv_provider; for every L-block the library calls
 *                     fill(ctx, L0, nl, dst, stream), which must enqueue on `stream` (a cudaStream_t) work that writes
 *                     B_vv[L0 .. L0+nl) as dst[nl][v][v] (device memory) and return 0.  Called in increasing L0, from
 *                     the calling thread, before thc_residual returns.                                            */
typedef enum { THC_BVV_DEVICE = 0, THC_BVV_HOST = 1, THC_BVV_PROVIDER = 2 } thc_bvv_mode;
typedef int (*thc_bvv_fill_fn)(void* ctx, int64_t L0, int64_t nl, double* dst_device, void* cuda_stream);
typedef struct { thc_bvv_fill_fn fill; void* ctx; } thc_bvv_provider;

/* Bits of thc_options.term_mask (terms to evaluate; 0 means all). */
enum { THC_TERM_S1 = 1, THC_TERM_S2 = 2, THC_TERM_S3 = 4, THC_TERM_S6 = 8, THC_TERM_S7 = 16, THC_TERM_S9 = 32,
       THC_TERM_ALL = 63 };

typedef struct {
  int64_t bL;               /* Cholesky vectors per L-block of the Alg.1/2/3/8 loop (0 = auto)              */
  int64_t bP7;              /* amplitude-grid rows per block of Alg.7 (0 = auto)                            */
  int64_t bX;               /* amplitude-grid rows per block of Alg.6 (0 = auto; rounded up to 16)          */
  int64_t bI;               /* ERI-grid points per chunk of Alg.6 (0 = auto)                                */
  int64_t workspace_bytes_max; /* cap for the auto block-size choice (0 = 92 % of free device memory)       */
  int64_t tma_min_flop;     /* GEMMs of at least this many flop with 16-byte aligned K-major operands run on the   */
                            /* TMA-fed persistent kernel, smaller ones on the cp.async kernel (0 = default 2e8,     */
                            /* -1 = never; tests use 1 to exercise the TMA kernel on small ragged shapes)           */
  int32_t term_mask;        /* THC_TERM_* bits, 0 = all                                                     */
  int32_t device;           /* CUDA device ordinal, -1 = current device                                     */
  int32_t bvv_mode;         /* thc_bvv_mode: what the B_vv argument of thc_residual[_terms] is                  */
  int32_t check_symmetry;   /* debug: non-zero = every residual call first verifies, in one extra pass over HBM  */
                            /* and one host synchronisation, that Z, V, every B^L_oo and (resident B_vv only)    */
                            /* every B^L_vv are symmetric to 1e-12 of their largest element; an unsymmetric      */
                            /* input makes the call return THC_ERR_INVALID_ARG instead of a silently wrong R     */
  int32_t use_graph;        /* 1 = capture the evaluation into a CUDA graph on first use and replay it while the */
                            /* pointers stay the same (launch-bound small shapes); 0 = never; -1 = auto: on when */
                            /* the shape is launch-bound (< 2e10 algorithmic flop) and B_vv is resident          */
  int32_t t2sq_algorithm;   /* how the ladder-type T2^2 terms (sigma6, Eqs.32+33) are evaluated: 4 = the O(N^4) Alg.6  */
                            /* (THC ERIs + the line-11 kernel), 5 = the O(N^5) GEMM-only Alg.4 + Alg.5, 0 = auto: the */
                            /* cheaper one by a flop/rate model ("ideally one would ..."); sharded      */
                            /* evaluations always use Alg.6                                                          */
} thc_options;

/* Create a handle for one problem shape.  (o, v, NL, NP, NX) as in BASELINE.json / PAPER.md l.47-54
 * (N_o, N_v, N_CD, N_aux, N_THC).  `opt` may be NULL.  Chooses block sizes, computes the workspace size. */
int thc_setup(thc_handle** h, int64_t o, int64_t v, int64_t NL, int64_t NP, int64_t NX, const thc_options* opt);
int thc_destroy(thc_handle* h);

/* Workspace the device-pointer entry points need (bytes); thc_workspace_bytes_host: what thc_residual_host
 * needs (the same plus staging copies of every input and of R).  A caller may provide a device buffer of at least
 * that size (256-byte aligned; it stays owned by the caller and must outlive every call that uses the handle);
 * otherwise the library allocates one with cudaMalloc on first use and frees it in thc_destroy. */
int64_t thc_workspace_bytes(const thc_handle* h);
int64_t thc_workspace_bytes_host(const thc_handle* h);
int thc_set_workspace(thc_handle* h, void* device_ptr, int64_t bytes);
/* CUDA stream (a cudaStream_t passed as void*) all work of this handle is enqueued on. */
int thc_set_stream(thc_handle* h, void* cuda_stream);

/* Block sizes actually in use: out[0..3] = bL, bP7, bX, bI. */
int thc_get_blocks(const thc_handle* h, int64_t out[4]);

/* R_PQ (device pointers; asynchronous).  Argument order follows the north_star:
 * thc_residual(X^o, X^v, Z, B_ov, B_oo, B_vv, Y, V, eps) -> R_PQ.
 * B_vv is typed const void* because its meaning depends on thc_options.bvv_mode: THC_BVV_DEVICE a device pointer
 * (const double*) to B_vv[NL][v][v]; THC_BVV_HOST a host pointer (const double*) to the same array; THC_BVV_PROVIDER
 * a const thc_bvv_provider*.  The same holds for thc_residual_terms and thc_residual_shard (there: the rank's own
 * slice, or, for a provider, the global L index is passed to fill); thc_residual_host takes a host array in the first
 * two modes and a provider in the third.                                                               */
int thc_residual(thc_handle* h, const double* Xo, const double* Xv, const double* Z, const double* B_ov,
                 const double* B_oo, const void* B_vv, const double* Y, const double* V, const double* eps,
                 double* R);

/* As thc_residual, and also writes each term separately (device pointers, any of them may be NULL):
 * terms[0..5] = sigma1, sigma2, sigma3, sigma6, sigma7, sigma9, each [NP][NP];  xi_oo[o][o] (Eq.39 l.280),
 * xi_vv[v][v] (Eq.40 l.283).  R may be NULL.                                                            */
int thc_residual_terms(thc_handle* h, const double* Xo, const double* Xv, const double* Z, const double* B_ov,
                       const double* B_oo, const void* B_vv, const double* Y, const double* V,
                       const double* eps, double* R, double* const terms[6], double* xi_oo, double* xi_vv);

/* T1-dressed evaluation: a complete CCSD residual.  With singles amplitudes t1[o][v] every Cholesky
 * vector is dressed, B^ = Xp^T B Xh with Xp = 1 - t1 (occupied rows, virtual columns), Xh = 1 + t1^T (Eqs.25-27; in the
 * MO basis the caller's B_oo, B_ov, B_vv are the BARE symmetric blocks, the library dresses them block by block and
 * B^_vo != B^_ov^T), the Fock matrix becomes F^ = Xp^T h Xh + sum_k [2 (pq|kk)^ - (pk|kq)^] (h fixed by the bare Fock
 * matrix being diag(eps)), and besides the doubles residual R_PQ (Eqs.28-41 with hatted integrals; the THC <ov|ov> terms
 * are untouched because B^_ia = B_ia) the singles residual
 *     sigma[o][v] = Omega G + Omega H (Eq.38 l.277; Alg.8 lines 11-12) + Omega I + Omega J (Eq.42 l.295; Alg.10)
 * is returned (unprojected, as the paper's algorithms produce it).  The symmetric-product shortcuts of the half-transforms
 * are switched off (only bra-ket symmetry is left, l.211); sigma1 stays symmetric.  terms[6] / sigma_terms[2] (G+H, I+J) /
 * xi_oo / xi_vv are optional outputs (NULL allowed).  Needs thc_workspace_bytes_t1(h) bytes of workspace, all terms
 * enabled (term_mask 0), and is evaluated on one device.  B_vv as in thc_residual. */
int64_t thc_workspace_bytes_t1(const thc_handle* h);
int thc_residual_t1(thc_handle* h, const double* Xo, const double* Xv, const double* Z, const double* t1,
                    const double* B_ov, const double* B_oo, const void* B_vv, const double* Y, const double* V,
                    const double* eps, double* R, double* sigma, double* const terms[6], double* const sigma_terms[2],
                    double* xi_oo, double* xi_vv);

/* Rank-reduced working variables (Eqs.13-14 l.116-120, Eq.22 l.178-181): with the orthogonalised CP factor
 * tau[NR][NP] (tau~^{PW}, P < NR) and the symmetric core T[NR][NR] in the semi-unitary basis,
 *     Z = tau^T T tau                (the THC-basis core T^{WX} of Eq.22),
 *     R_rr = tau R(Z) tau^T          (the amplitude equations projected with U~ = sum_W y y tau~, Eqs.6 and 14).
 * Device pointers, asynchronous.  Z_out[NP][NP] (optional, may be NULL) receives Z.  Needs thc_workspace_bytes_rr(h, NR)
 * bytes of workspace (the residual's plus Z, R and one NR x NP temporary).  The other arguments are thc_residual's. */
int64_t thc_workspace_bytes_rr(const thc_handle* h, int64_t NR);
int thc_residual_rr(thc_handle* h, int64_t NR, const double* tau, const double* T, const double* Xo, const double* Xv,
                    const double* B_ov, const double* B_oo, const void* B_vv, const double* Y, const double* V,
                    const double* eps, double* R_rr, double* Z_out);

/* Correlation energy E = sum_L [ 2 a^L.Z.a^L - sum_PQ Z_PQ E^L_PQ E^L_QP ] (factorised form of
 * sum (2t - t^x)(ia|jb); a^L, E^L from Alg.8 l.5-6).  Device pointers in, one double written to the HOST
 * address E_host; synchronises the stream.                                                             */
int thc_energy(thc_handle* h, const double* Xo, const double* Xv, const double* Z, const double* B_ov,
               double* E_host);

/* As thc_energy but asynchronous: E is written to the DEVICE address E_dev; no synchronisation. */
int thc_energy_device(thc_handle* h, const double* Xo, const double* Xv, const double* Z, const double* B_ov,
                      double* E_dev);

/* ---- Sharded evaluation over several devices (one handle per device) -----
 * The Cholesky index is cut into equal contiguous ranges (Alg.1/2/3/8 partial sums) and the amplitude-grid rows of the
 * T2^2 terms (Alg.6/7) into equal contiguous row blocks:  thc_shard_range(NL, NP, rank, nranks, out) writes
 * out = {L_begin, L_end, P_begin, P_end} (needs no device).
 *   1. every rank calls thc_residual_shard with B_ov, B_oo, B_vv pointing at ITS OWN slice (vector L_begin first; the
 *      slice may be empty, the pointers are then ignored) and a device buffer `packed` of thc_shard_doubles() doubles:
 *      [sigma1 | sigma2 | C3 | sigma6 rows | sigma7 rows | C7 rows | xi_oo | xi_vv], rows of other ranks zero;
 *   2. the caller sums `packed` element-wise over the ranks (one all-reduce; that is the only exchange step);
 *   3. every rank calls thc_residual_finish with the summed buffer (it is modified): Alg.3 tail, Alg.9, the
 *      C7 V C7^T part of Alg.7 and the final sum give R (and, if terms != NULL, each term; any entry may be NULL).
 * thc_energy_shard writes the rank's partial energy (its Cholesky range) to E_dev; the caller sums over ranks. */
int thc_shard_range(int64_t NL, int64_t NP, int rank, int nranks, int64_t out[4]);
int64_t thc_shard_doubles(const thc_handle* h);
int thc_residual_shard(thc_handle* h, const double* Xo, const double* Xv, const double* Z, const double* B_ov,
                       const double* B_oo, const void* B_vv, const double* Y, const double* V, const double* eps,
                       int rank, int nranks, double* packed);
int thc_residual_finish(thc_handle* h, const double* Xo, const double* Xv, const double* Z, const double* Y,
                        const double* V, const double* eps, double* packed, double* R, double* const terms[6]);
int thc_energy_shard(thc_handle* h, const double* Xo, const double* Xv, const double* Z, const double* B_ov, int rank,
                     int nranks, double* E_dev);

/* End-to-end entry with HOST buffers: copies every input host->device on the handle's stream, evaluates
 * R (and E if E_host != NULL), copies R device->host into R_host[NP][NP], synchronises.  The staging
 * buffers are part of the workspace (thc_workspace_bytes_host includes them).                       */
int thc_residual_host(thc_handle* h, const double* Xo, const double* Xv, const double* Z, const double* B_ov,
                      const double* B_oo, const void* B_vv, const double* Y, const double* V,
                      const double* eps, double* R_host, double* E_host);

/* Number of kernels this handle has launched since creation (its own kernels only; no library calls). */
int64_t thc_kernel_launches(const thc_handle* h);
/* Algorithmic FP64 flop count of one residual evaluation for this shape (SURVEY.md 8(a) formulas). */
double thc_algorithmic_flops(const thc_handle* h);

/* Per-class kernel timing for roofline measurement.  After thc_profile_begin every kernel launch of a class
 * whose bit is set in class_mask is bracketed by CUDA events on the handle's stream (bit 0: DMMA GEMM incl. its
 * split-K reduction, bit 1: Alg.6 line 11 triple product, bit 2: Hadamard / reduction kernels).
 * thc_profile_end synchronises the stream, returns the summed device time (milliseconds) and the number of timed
 * launches per class, and switches the timing off again.  Not for use while the stream is being captured. */
int thc_profile_begin(thc_handle* h, int class_mask);
int thc_profile_end(thc_handle* h, double ms[3], int64_t counts[3]);
/* Work of the launches timed by the last thc_profile_end, per class: EXECUTED flop for classes 0 and 1 (every GEMM
 * launched, recomputation included; 5 flop per (P,Q,R,I) of line 11 over the padded extents), algorithmic HBM bytes
 * (each operand element read once, each result written once) for class 2. */
int thc_profile_work(const thc_handle* h, double work[3]);
/* Per-launch records of the last thc_profile_end, in launch order: thc_profile_launches returns how many there are;
 * thc_profile_launch copies record k: its class (0, 1, 2 as above), its device time in milliseconds, its work (as in
 * thc_profile_work) and a NUL-terminated description (kernel, shape, tile) truncated to desc_bytes.  Any out pointer
 * may be NULL. */
int64_t thc_profile_launches(const thc_handle* h);
int thc_profile_launch(const thc_handle* h, int64_t k, int* cls, double* ms, double* work, char* desc,
                       int64_t desc_bytes);
/* ALGORITHMIC work of one residual evaluation per kernel class (SURVEY.md 8(a) formulas; no symmetry savings, no
 * recomputation, no padding): work[0] = flop of every GEMM-shaped step (H0-H2, H4-H10 without line 11), work[1] =
 * 5 NX NP^3 flop of Alg.6 line 11, work[2] = 5 NL NP^2 flop of the H3 Hadamard combine.  Their sum is
 * thc_algorithmic_flops. */
int thc_algorithmic_work(const thc_handle* h, double work[3]);

/* Bare FP64 DMMA GEMM of the library (the kernel every GEMM chain uses), exposed for tests and roofline
 * measurement:  C[M][N] = alpha * sum_k A(m,k) B(n,k) + beta * C,  A(m,k) = A[m*lda+k] if a_kmajor else
 * A[k*lda+m];  B(n,k) = B[n*ldb+k] if b_kmajor else B[k*ldb+n].  Device pointers, asynchronous.        */
int thc_dgemm(thc_handle* h, int a_kmajor, int b_kmajor, int64_t M, int64_t N, int64_t K, double alpha,
              const double* A, int64_t lda, const double* B, int64_t ldb, double beta, double* C, int64_t ldc);

/* Alg.6 line 11 (l.714) alone, for tests and roofline measurement:
 * H[p][q][r] (+)= sum_I (E[I][p][q] F[I][p][r] + E[I][p][r] F[I][p][q]) G[I][q][r]
 * E, F: [nI][nPp][NPp], G: [nI][NPp][NPp], H: [nPp][NPp][NPp]; NPp a multiple of 32, nPp of 16 (padded extents;
 * padded entries are computed from whatever the padding holds and must be ignored).  All pointers 16-byte aligned. */
int thc_triple_product(thc_handle* h, int64_t nI, int64_t nPp, int64_t NPp, const double* E, const double* F,
                       const double* G, double* H, int accumulate);

/* Measured FP64 / shared-memory ceilings of the handle's device (synchronous; ~0.3 s).  MEASURED_PEAKS.json has no
 * FP64 entry, so the rooflines of DESIGN.md section 7 rest on these:  out[0] issue rate of the FP64 tensor instruction
 * (mma.sync.m8n8k4.f64 = SASS DMMA.8x8x4) in TFLOP/s, out[1] DFMA issue rate in TFLOP/s, out[2] both interleaved 1:1 in
 * one warp (sum of both, TFLOP/s; ~ out[0] means one shared pipe), out[3], out[4], out[5] shared memory -> register
 * bandwidth with 4-, 8- and 16-byte conflict-free loads in bytes per clock per SM at the maximum SM clock, out[6] that
 * clock in MHz, out[7] = 0. */
int thc_probe(thc_handle* h, double out[8]);

/* ---- second workload: the two O(N^4) set-up steps of PAPER.md's appendices, on the same kernels ----
 *
 * thc_mp2_density: MP2 one-particle density matrix from THC-factorised doubles, Appendix II (l.375-415):
 *   D_oo[i][j] = -2 sum_kab t_ik^ab (2 t_jk^ab - t_jk^ba)   (Eq.47),   D_vv[a][b] = 2 sum_ijc t_ij^ac (2 t_ij^bc - t_ji^bc)   (Eq.48)
 * with t_ij^ab = sum_PQ Xo[i,P] Xv[a,P] Z[P,Q] Xo[j,Q] Xv[b,Q] (Eq.23), evaluated in the O(N^4) factorisation of
 * Eqs.51-56.  Xo [o][NP], Xv [v][NP], Z [NP][NP] (need not be symmetric), D_oo [o][o], D_vv [v][v]: device pointers,
 * row-major, caller-owned; o, v, NP are the handle's.  Asynchronous on the handle's stream.  Needs
 * thc_workspace_bytes_mp2 bytes of workspace (grown like thc_residual's when the library owns it, THC_ERR_NO_MEMORY when a
 * caller-provided one is too small). */
int64_t thc_workspace_bytes_mp2(const thc_handle* h);
int thc_mp2_density(thc_handle* h, const double* Xo, const double* Xv, const double* Z, double* D_oo, double* D_vv);

/* thc_cp_als_update: one alternating-least-squares factor update of a CP factorisation A_ijk ~ sum_n X_i^n Y_j^n Z_k^n
 * (Appendix I, l.355-373): S of Eq.45, R of Eq.46, then `iters` iterations of the conjugate gradient method
 * preconditioned with diag(S) on S x_i = R_i (Eq.44) for every row i, started from the X passed in (R22).
 * A [I][J][K], Y [J][N], Z [K][N]: inputs; X [I][N]: in = starting guess, out = updated factor; rnorm2 [I] or NULL:
 * |R_i - S x_i|^2 of the recurrence residual after the last iteration.  Device pointers, row-major, caller-owned;
 * J * K < 2^31.  The sizes are independent of the handle's (it supplies device, stream and workspace:
 * thc_workspace_bytes_als bytes).  The other two factors are updated by the same call on the permuted array (the paper
 * keeps the three permutations of A resident, l.373).  Rows are independent (l.373): a multi-GPU update gives every
 * rank a block of rows, A[i0:i1] and X[i0:i1], and the whole Y and Z -- no exchange inside the call, S is formed
 * redundantly as in the paper; the caller gathers the updated rows.  Asynchronous. */
int64_t thc_workspace_bytes_als(const thc_handle* h, int64_t I, int64_t J, int64_t K, int64_t N);
int thc_cp_als_update(thc_handle* h, int64_t I, int64_t J, int64_t K, int64_t N, const double* A, const double* Y,
                      const double* Z, double* X, int iters, double* rnorm2);

/* ---- allocation-free entry point ------------------------------------------------------------------------------------
 * For callers that cannot call cudaMalloc (code under CUDA-graph capture, tight serving loops, harnesses that forbid
 * it): the split-K FP64 DMMA GEMM of the GEMM chains ("rate limiting step"; same kernels as thc_dgemm)
 * with the split-K partial tiles in a static device array of THC_STATIC_SCRATCH_BYTES instead of a workspace.  Needs no
 * thc_handle and calls no cudaMalloc / cudaFree / allocating library routine.
 *
 *   C[M][N] = alpha * sum_k A[m*lda + k] * B[n*ldb + k] + beta * C          (both operands K-major, row-major C)
 *
 * A, B, C: device pointers on `device` (-1 = the current device), 8-byte aligned (16-byte aligned with even lda / ldb
 * selects the faster copy path), not overlapping; caller-owned.  `stream`: a cudaStream_t (NULL = default stream); the
 * call is asynchronous.  `splits`: number of K ranges, >= 1, or 0 = chosen by the library (about two waves of CTAs,
 * within the scratch limit).  With splits S the call needs S * M * N * 8 bytes of scratch: more than
 * THC_STATIC_SCRATCH_BYTES returns THC_ERR_STATIC_LIMIT (nothing is launched); splits = 0 never exceeds the limit (it
 * falls back to fewer splits, down to 1 = no scratch).  splits > 1 is summed in split order (deterministic).
 *
 * The array is one per GPU per process, held from library load until exit, and shared by every call: two calls that
 * overlap on the GPU (different streams, or graphs replayed concurrently) race on it; calls on one stream do not.  It
 * keeps the previous call's partial tiles; nothing has to start at zero because every partial element that the
 * reduction reads is written by the GEMM kernel of the same call first.
 *
 * thc_static_init(device) does the once-per-device set-up (address of the array, shared-memory opt-in of the kernels,
 * SM count) ahead of time, e.g. before a graph capture; thc_dgemm_static does it on first use otherwise.          */
#define THC_STATIC_SCRATCH_BYTES (16ll << 20)
int thc_static_init(int device);
int thc_dgemm_static(int device, void* stream, int64_t M, int64_t N, int64_t K, int splits, double alpha,
                     const double* A, int64_t lda, const double* B, int64_t ldb, double beta, double* C, int64_t ldc);

const char* thc_strerror(int status);
int thc_last_error(const thc_handle* h);       /* the cudaError_t of the last THC_ERR_CUDA on this handle, else 0 */
int thc_last_cuda_error(const thc_handle* h);   /* older name of thc_last_error (same value)                       */

#ifdef __cplusplus
}
#endif
#endif /* THC_H_ */
