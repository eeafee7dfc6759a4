"""Counter-based, order-free generators for the five synthetic workloads.

Every scalar drawn is a pure function of (seed, tensor_id, flat_index):

    h      = splitmix64(splitmix64(seed * 2^32 + tensor_id) + flat_index)   (uint64)
    u(h)   = ((h >> 11) + 0.5) * 2^-53                                      in (0, 1)
    normal = sqrt(-2 ln u(h1)) * cos(2 pi u(h2)),  h1 = mix(2 idx), h2 = mix(2 idx + 1)

so any block of any tensor can be produced independently (needed for the
paper-scale config, whose B_vv is ~304 GB and is only ever materialised in
L-blocks).  Distributions follow BASELINE.json `configs` with the readings
R15-R17 of SURVEY.md section 8(c):

    eps_o ~ U[-1.5, -0.3], eps_v ~ U[0.1, 3.0]      (sorted ascending)
    Xo [o, NP], Xv [v, NP]      ~ N(0,1) / sqrt(NP)
    Z  [NP, NP]                 = 0.1 * (G + G^T) / 2,   G ~ N(0,1)
    B^L [(o+v), (o+v)]          = (G_L + G_L^T) / 2 * exp(-L / lambda),  lambda = NL / 4
    Y  [(o+v), NX]              ~ N(0,1) / sqrt(NX)
    V  [NX, NX]                 = G G^T / NX,  G ~ N(0,1)   (symmetric PSD)

The paper measures on real molecules that are not
available here; these seeded tensors take over their shapes only.
"""
from __future__ import annotations

from dataclasses import dataclass
import numpy as np

# (o, v, NL, NP, NX), seed = config index  -- BASELINE.json `configs`
CONFIGS = {
    0: dict(o=5, v=20, NL=60, NP=50, NX=100, seed=0),
    1: dict(o=20, v=100, NL=360, NP=300, NX=600, seed=1),
    2: dict(o=60, v=340, NL=1200, NP=1000, NX=2000, seed=2),
    3: dict(o=150, v=850, NL=3000, NP=2500, NX=5000, seed=3),
    4: dict(o=250, v=2250, NL=7500, NP=5000, NX=10000, seed=4),
}

TENSOR_IDS = dict(eps_o=0, eps_v=1, Xo=2, Xv=3, Z=4, B=5, Y=6, VG=7)

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _splitmix64(x: np.ndarray) -> np.ndarray:
    """splitmix64 finaliser on uint64 arrays (wrap-around arithmetic)."""
    with np.errstate(over="ignore"):
        z = (x + np.uint64(0x9E3779B97F4A7C15)) & _M64
        z = ((z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)) & _M64
        z = ((z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)) & _M64
        return z ^ (z >> np.uint64(31))


def _key(seed: int, tensor_id: int) -> np.uint64:
    k = np.array([(int(seed) << 32) + int(tensor_id)], dtype=np.uint64)
    return _splitmix64(k)[0]


def _u01(h: np.ndarray) -> np.ndarray:
    return ((h >> np.uint64(11)).astype(np.float64) + 0.5) * (2.0 ** -53)


def uniform_block(seed: int, tensor_id: int, flat_index: np.ndarray) -> np.ndarray:
    """U(0,1) draws at the given flat indices (any shape, any order)."""
    idx = np.asarray(flat_index, dtype=np.uint64)
    with np.errstate(over="ignore"):
        h = _splitmix64(_key(seed, tensor_id) + idx)
    return _u01(h)


def normal_block(seed: int, tensor_id: int, flat_index: np.ndarray) -> np.ndarray:
    """N(0,1) draws (Box-Muller, cosine branch) at the given flat indices."""
    idx = np.asarray(flat_index, dtype=np.uint64)
    key = _key(seed, tensor_id)
    with np.errstate(over="ignore"):
        h1 = _splitmix64(key + np.uint64(2) * idx)
        h2 = _splitmix64(key + np.uint64(2) * idx + np.uint64(1))
    return np.sqrt(-2.0 * np.log(_u01(h1))) * np.cos(2.0 * np.pi * _u01(h2))


def _normal_full(seed, tensor_id, shape, chunk=1 << 22):
    n = int(np.prod(shape))
    out = np.empty(n, dtype=np.float64)
    for s in range(0, n, chunk):
        e = min(n, s + chunk)
        out[s:e] = normal_block(seed, tensor_id, np.arange(s, e, dtype=np.uint64))
    return out.reshape(shape)


def config_dims(cfg: int):
    c = CONFIGS[cfg]
    return c["o"], c["v"], c["NL"], c["NP"], c["NX"]


def _bsym_block(seed, n, NL, L0, L1, p0, p1, q0, q1):
    """Rows p0:p1, cols q0:q1 of B^L = (G_L + G_L^T)/2 * exp(-L/lambda), L in [L0, L1)."""
    lam = NL / 4.0
    L = np.arange(L0, L1, dtype=np.uint64)[:, None, None]
    p = np.arange(p0, p1, dtype=np.uint64)[None, :, None]
    q = np.arange(q0, q1, dtype=np.uint64)[None, None, :]
    nn = np.uint64(n)
    g1 = normal_block(seed, TENSOR_IDS["B"], (L * nn + p) * nn + q)
    g2 = normal_block(seed, TENSOR_IDS["B"], (L * nn + q) * nn + p)
    scale = np.exp(-np.arange(L0, L1, dtype=np.float64) / lam)[:, None, None]
    return 0.5 * (g1 + g2) * scale


def bvv_block(seed: int, o: int, v: int, NL: int, L0: int, L1: int) -> np.ndarray:
    """B_vv[L0:L1] as a [L1-L0, v, v] array without forming anything else."""
    return _bsym_block(seed, o + v, NL, L0, L1, o, o + v, o, o + v)


class LazyCholesky:
    """B_oo ("oo") or B_ov ("ov") of a workload as an array-like that draws the requested Cholesky vectors on demand:
    `.shape` and `[L0:L1]` only (what an L-blocked consumer needs).  At config 4 B_ov alone is 34 GB; a consumer that
    walks the vectors block by block never has to hold it."""

    def __init__(self, seed, o, v, NL, kind):
        self.seed, self.o, self.v, self.NL, self.kind = seed, o, v, NL, kind
        self.shape = (NL, o, o if kind == "oo" else v)

    def __getitem__(self, key):
        if not isinstance(key, slice) or key.step not in (None, 1):
            raise IndexError("LazyCholesky supports contiguous slices of the Cholesky index only")
        L0, L1, _ = key.indices(self.NL)
        o, n = self.o, self.o + self.v
        q0, q1 = (0, o) if self.kind == "oo" else (o, n)
        return np.ascontiguousarray(_bsym_block(self.seed, n, self.NL, L0, L1, 0, o, q0, q1))


@dataclass
class ThcInputs:
    o: int
    v: int
    NL: int
    NP: int
    NX: int
    seed: int
    eps: np.ndarray    # [o+v], occupied first
    Xo: np.ndarray     # [o, NP]
    Xv: np.ndarray     # [v, NP]
    Z: np.ndarray      # [NP, NP] symmetric
    B_oo: np.ndarray   # [NL, o, o]
    B_ov: np.ndarray   # [NL, o, v]
    B_vv: np.ndarray   # [NL, v, v]  (None when with_bvv=False)
    Y: np.ndarray      # [o+v, NX]
    V: np.ndarray      # [NX, NX] symmetric PSD

    @property
    def Yo(self):
        return self.Y[: self.o]

    @property
    def Yv(self):
        return self.Y[self.o:]

    def nbytes(self):
        return sum(a.nbytes for a in (self.eps, self.Xo, self.Xv, self.Z, self.B_oo, self.B_ov,
                                      self.Y, self.V) ) + (0 if self.B_vv is None else self.B_vv.nbytes)


def make_inputs(o, v, NL, NP, NX, seed, with_bvv=True, z_scale=0.1, l_keep=None) -> ThcInputs:
    """Draw one full input set.  `z_scale` is the std of Z before symmetrisation (R15).  `l_keep` draws only the first
    l_keep Cholesky vectors of the NL (same values as in the full set; a bounded sample of a large workload)."""
    n = o + v
    NL_full, NL = NL, (NL if l_keep is None else min(NL, int(l_keep)))
    eps_o = np.sort(-1.5 + 1.2 * uniform_block(seed, TENSOR_IDS["eps_o"], np.arange(o)))
    eps_v = np.sort(0.1 + 2.9 * uniform_block(seed, TENSOR_IDS["eps_v"], np.arange(v)))
    eps = np.concatenate([eps_o, eps_v])
    Xo = _normal_full(seed, TENSOR_IDS["Xo"], (o, NP)) / np.sqrt(NP)
    Xv = _normal_full(seed, TENSOR_IDS["Xv"], (v, NP)) / np.sqrt(NP)
    G = _normal_full(seed, TENSOR_IDS["Z"], (NP, NP))
    Z = z_scale * 0.5 * (G + G.T)
    del G
    B_oo = np.ascontiguousarray(_bsym_block(seed, n, NL_full, 0, NL, 0, o, 0, o))
    B_ov = np.ascontiguousarray(_bsym_block(seed, n, NL_full, 0, NL, 0, o, o, n))
    B_vv = None
    if with_bvv:
        B_vv = np.empty((NL, v, v), dtype=np.float64)
        step = max(1, (1 << 22) // max(1, v * v))
        for L0 in range(0, NL, step):
            L1 = min(NL, L0 + step)
            B_vv[L0:L1] = bvv_block(seed, o, v, NL_full, L0, L1)
    Y = _normal_full(seed, TENSOR_IDS["Y"], (n, NX)) / np.sqrt(NX)
    G = _normal_full(seed, TENSOR_IDS["VG"], (NX, NX))
    V = (G @ G.T) / NX
    V = 0.5 * (V + V.T)
    return ThcInputs(o, v, NL, NP, NX, seed, eps, Xo, Xv, Z, B_oo, B_ov, B_vv, Y, V)


def make_config(cfg: int, with_bvv=True) -> ThcInputs:
    c = CONFIGS[cfg]
    return make_inputs(c["o"], c["v"], c["NL"], c["NP"], c["NX"], c["seed"], with_bvv=with_bvv)
