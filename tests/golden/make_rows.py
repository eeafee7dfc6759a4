#!/usr/bin/env python
"""Writes stored expected rows R[P, :] of the residual terms at a BASELINE config -- calls only oracle/ and thc_synth/.

    python tests/golden/make_rows.py --config 4 --row 2718 --terms s1,s2,s3,s7 [--lblock 4] [--outdir tests/golden]

One text file per term, tests/golden/config<C>_row<P>_<term>.txt: '#' header lines (what, how, when), then the NP values
as C99 hex floats (exact).  At config 4 one row of sigma1..sigma3 takes hours of CPU and one of sigma6 about as long, more
than a GPU-box call may last, so tests/test_gpu_rows.py reads these files when they exist instead of recomputing the rows
next to the GPU evaluation.  The inputs are the seeded CPU generators of thc_synth (the GPU test draws the same tensors on
the device: uniforms bit-identical, normals equal to an ulp or two, V = G G^T / NX by another matmul -- differences
far below the 1e-10 tolerance).  Nothing here comes from the CUDA path.
"""
import argparse
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

LINEAR_IN_B = ("s1", "s2", "s3")          # need the Cholesky vectors; the others only Xo, Xv, Z, Y, V, eps


def row_file(outdir, cfg, P, term):
    return os.path.join(outdir, f"config{cfg}_row{P}_{term}.txt")


def load_rows(outdir, cfg, P):
    """{term: row} for every stored term of (cfg, P)."""
    out = {}
    for term in ("s1", "s2", "s3", "s6", "s7", "s9"):
        path = row_file(outdir, cfg, P, term)
        if os.path.exists(path):
            with open(path) as f:
                vals = [float.fromhex(tok) for line in f if not line.startswith("#") for tok in line.split()]
            out[term] = np.array(vals)
    return out


def main():
    from oracle.rows import RowOracle
    from thc_synth import CONFIGS, LazyCholesky, bvv_block, make_inputs
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, required=True)
    ap.add_argument("--row", type=int, required=True)
    ap.add_argument("--terms", required=True, help="comma-separated subset of s1,s2,s3,s6,s7 (sigma9 needs the full xi)")
    ap.add_argument("--lblock", type=int, default=4)
    ap.add_argument("--bvv-on-gpu", action="store_true",
                    help="draw the B_vv blocks with thc_synth.device on cuda:0 (same seeded function, values equal to an ulp or "
                         "two); the numpy generator needs ~1 s per vector at config 4, i.e. hours per row")
    ap.add_argument("--outdir", default=os.path.dirname(os.path.abspath(__file__)))
    args = ap.parse_args()
    terms = tuple(args.terms.split(","))
    os.makedirs(args.outdir, exist_ok=True)
    assert all(t in ("s1", "s2", "s3", "s6", "s7") for t in terms), terms
    c = CONFIGS[args.config]
    o, v, NL, NP, NX, seed = c["o"], c["v"], c["NL"], c["NP"], c["NX"], c["seed"]
    t0 = time.perf_counter()
    x = make_inputs(o, v, NL, NP, NX, seed, with_bvv=False, l_keep=1)          # factors, grid, eps; one Cholesky vector
    if any(t in LINEAR_IN_B for t in terms):                                  # the Cholesky vectors, drawn block by block
        B_ov, B_oo = LazyCholesky(seed, o, v, NL, "ov"), LazyCholesky(seed, o, v, NL, "oo")
        B_vv = lambda L0, L1: bvv_block(seed, o, v, NL, L0, L1)
        if args.bvv_on_gpu:
            from thc_synth import device as synth
            B_vv = lambda L0, L1: synth.bvv_block(seed, o, v, NL, L0, L1, "cuda").cpu().numpy()
    else:
        B_ov, B_oo, B_vv = x.B_ov, x.B_oo, np.zeros((1, v, v))
    print(f"inputs drawn in {time.perf_counter() - t0:.0f} s", flush=True)
    ro = RowOracle(x.Xo, x.Xv, x.Z, B_ov, B_oo, B_vv, x.Y, x.V, x.eps, lblock=args.lblock)
    for term in terms:
        t0 = time.perf_counter()
        row = ro.row(args.row, terms=(term,))[term]
        dt = time.perf_counter() - t0
        path = row_file(args.outdir, args.config, args.row, term)
        with open(path, "w") as f:
            f.write(f"# R[P={args.row}, :] of term {term}, BASELINE config {args.config} (o={o} v={v} NL={NL} NP={NP} NX={NX}, seed {seed})\n")
            f.write(f"# written by tests/golden/make_rows.py from oracle/rows.py (RowOracle.row, lblock={args.lblock}"
                    f"{', B_vv blocks drawn by thc_synth.device' if args.bvv_on_gpu and term in ('s1', 's3') else ''}) in {dt:.0f} s CPU, "
                    f"{time.strftime('%Y-%m-%d')}; C99 hex floats\n")
            for k in range(0, NP, 4):
                f.write(" ".join(float(val).hex() for val in row[k:k + 4]) + "\n")
        print(f"{term}: {dt:.0f} s CPU -> {path}", flush=True)


if __name__ == "__main__":
    main()
