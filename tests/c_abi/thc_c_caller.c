/* A plain-C caller of the library (C99; no CUDA headers, no torch): reads one input set from a binary file of doubles,
 * runs thc_setup -> thc_residual_host (R and E through host buffers) -> thc_destroy and writes R followed by E to the
 * output file.  tests/test_c_abi.py builds it with gcc against include/thc.h and libthc_b200.so and compares the result
 * with the CPU oracle (GPU test); the CPU suite only checks that it compiles and links.
 *
 *   thc_c_caller o v NL NP NX inputs.bin out.bin
 *   inputs.bin = Xo[o*NP] Xv[v*NP] Z[NP*NP] B_ov[NL*o*v] B_oo[NL*o*o] B_vv[NL*v*v] Y[(o+v)*NX] V[NX*NX] eps[o+v]  */
#include <stdio.h>
#include <stdlib.h>
#include "thc.h"

int main(int argc, char** argv) {
  if (argc != 8) { fprintf(stderr, "usage: %s o v NL NP NX inputs.bin out.bin\n", argv[0]); return 2; }
  const int64_t o = atoll(argv[1]), v = atoll(argv[2]), NL = atoll(argv[3]), NP = atoll(argv[4]), NX = atoll(argv[5]);
  const int64_t n[9] = {o * NP, v * NP, NP * NP, NL * o * v, NL * o * o, NL * v * v, (o + v) * NX, NX * NX, o + v};
  double* in[9];
  FILE* f = fopen(argv[6], "rb");
  if (!f) { perror("inputs"); return 2; }
  for (int k = 0; k < 9; k++) {
    in[k] = (double*)malloc((size_t)n[k] * sizeof(double));
    if (!in[k] || fread(in[k], sizeof(double), (size_t)n[k], f) != (size_t)n[k]) { fprintf(stderr, "short read\n"); return 2; }
  }
  fclose(f);
  double* R = (double*)malloc((size_t)(NP * NP + 1) * sizeof(double));
  thc_options opt = {0};
  opt.device = -1;
  opt.check_symmetry = 1;
  thc_handle* h = NULL;
  int st = thc_setup(&h, o, v, NL, NP, NX, &opt);
  if (st == THC_OK)
    st = thc_residual_host(h, in[0], in[1], in[2], in[3], in[4], in[5], in[6], in[7], in[8], R, &R[NP * NP]);
  if (st != THC_OK) {
    fprintf(stderr, "thc error %d: %s (cuda %d)\n", st, thc_strerror(st), h ? thc_last_error(h) : 0);
    return 1;
  }
  printf("launches %lld  workspace %lld bytes  E %.15e\n", (long long)thc_kernel_launches(h),
         (long long)thc_workspace_bytes_host(h), R[NP * NP]);
  thc_destroy(h);
  f = fopen(argv[7], "wb");
  if (!f || fwrite(R, sizeof(double), (size_t)(NP * NP + 1), f) != (size_t)(NP * NP + 1)) { perror("output"); return 2; }
  fclose(f);
  return 0;
}
