"""A C-language caller of the boundary: tests/c_abi/thc_c_caller.c includes include/thc.h, links libthc_b200.so and runs
setup -> residual (host buffers) -> energy -> destroy.  CPU suite: it compiles as C99 and links.  GPU suite: its R and E
on BASELINE config 0 match the dense oracle."""
import os
import subprocess

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "tests", "c_abi", "thc_c_caller.c")
NAMES = ("Xo", "Xv", "Z", "B_ov", "B_oo", "B_vv", "Y", "V", "eps")


def _build(tmp_path):
    import paper_2111_11473_b200 as thc
    thc.build()
    exe = str(tmp_path / "thc_c_caller")
    libdir = os.path.dirname(thc.LIB_PATH)
    cmd = ["gcc", "-std=c99", "-Wall", "-Werror", "-O1", "-I", os.path.join(ROOT, "include"), SRC, "-o", exe,
           "-L", libdir, "-l:libthc_b200.so", f"-Wl,-rpath,{libdir}"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    assert r.returncode == 0, r.stderr
    return exe


def test_c_caller_compiles_and_links(tmp_path):
    exe = _build(tmp_path)
    r = subprocess.run([exe], capture_output=True, text=True)        # no arguments: usage message, exit 2
    assert r.returncode == 2 and "usage" in r.stderr


@pytest.mark.gpu
def test_c_caller_matches_oracle(tmp_path, oracle_cfg):
    x, ref = oracle_cfg(0)
    exe = _build(tmp_path)
    inp, out = tmp_path / "in.bin", tmp_path / "out.bin"
    with open(inp, "wb") as f:
        for n in NAMES:
            f.write(np.ascontiguousarray(getattr(x, n), dtype=np.float64).tobytes())
    r = subprocess.run([exe, str(x.o), str(x.v), str(x.NL), str(x.NP), str(x.NX), str(inp), str(out)],
                       capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stdout + r.stderr
    res = np.fromfile(out, dtype=np.float64)
    R, E = res[:-1].reshape(x.NP, x.NP), res[-1]
    assert np.abs(R - ref["R"]).max() <= 1e-10 * np.abs(ref["R"]).max()
    assert abs(E - ref["E"]) <= 1e-9
