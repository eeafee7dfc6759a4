"""The same counter-based generators as generators.py, evaluated with torch ops on a CUDA device.

For BASELINE configs 3 and 4 the inputs are tens to hundreds of GB (B_vv: 17 GB / 304 GB); drawing them with numpy on
the host would take minutes to hours, so they are drawn where they are used.  Every scalar is the same function of
(seed, tensor_id, flat_index) as in generators.py (splitmix64 -> 53-bit uniform -> Box-Muller, cosine branch); the
uniforms are bit-identical to the numpy ones, the normals agree to the last ulp or two (CUDA's log/cos/sqrt vs libm).
Tests that compare against the CPU oracle at these sizes copy the very tensors produced here to the host, so both sides
see identical inputs.  This module holds none of the method's arithmetic and imports nothing of the library.
"""
from __future__ import annotations

import math

import torch

from .generators import CONFIGS, TENSOR_IDS

_MASK = (1 << 64) - 1


def _s64(x: int) -> int:
    """Python int (mod 2^64) -> the int64 with the same bit pattern."""
    x &= _MASK
    return x - (1 << 64) if x >= (1 << 63) else x


def _lsr(z: torch.Tensor, n: int) -> torch.Tensor:
    """Logical right shift of int64 bit patterns."""
    return (z >> n) & ((1 << (64 - n)) - 1)


def _splitmix64(x: torch.Tensor) -> torch.Tensor:
    z = x + _s64(0x9E3779B97F4A7C15)
    z = (z ^ _lsr(z, 30)) * _s64(0xBF58476D1CE4E5B9)
    z = (z ^ _lsr(z, 27)) * _s64(0x94D049BB133111EB)
    return z ^ _lsr(z, 31)


def _key(seed: int, tensor_id: int) -> int:
    z = ((int(seed) << 32) + int(tensor_id) + 0x9E3779B97F4A7C15) & _MASK
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _MASK
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _MASK
    return _s64(z ^ (z >> 31))


def _u01(h: torch.Tensor) -> torch.Tensor:
    return (_lsr(h, 11).to(torch.float64) + 0.5) * (2.0 ** -53)


def uniform_block(seed, tensor_id, idx: torch.Tensor) -> torch.Tensor:
    return _u01(_splitmix64(idx + _key(seed, tensor_id)))


def normal_block(seed, tensor_id, idx: torch.Tensor) -> torch.Tensor:
    key = _key(seed, tensor_id)
    u1 = _u01(_splitmix64(2 * idx + key))
    u2 = _u01(_splitmix64(2 * idx + (key + 1)))
    return torch.sqrt(-2.0 * torch.log(u1)) * torch.cos((2.0 * math.pi) * u2)


def _normal_full(seed, tensor_id, shape, device, chunk=1 << 26):
    n = math.prod(shape)
    out = torch.empty(n, dtype=torch.float64, device=device)
    for s in range(0, n, chunk):
        e = min(n, s + chunk)
        out[s:e] = normal_block(seed, tensor_id, torch.arange(s, e, dtype=torch.int64, device=device))
    return out.reshape(shape)


def bsym_block(seed, n, NL, L0, L1, p0, p1, q0, q1, device, out=None):
    """Rows p0:p1, cols q0:q1 of B^L = (G_L + G_L^T)/2 * exp(-L/lambda), lambda = NL/4, for L in [L0, L1)."""
    res = out if out is not None else torch.empty(L1 - L0, p1 - p0, q1 - q0, dtype=torch.float64, device=device)
    p = torch.arange(p0, p1, dtype=torch.int64, device=device)[:, None]
    q = torch.arange(q0, q1, dtype=torch.int64, device=device)[None, :]
    for L in range(L0, L1):                       # one vector at a time keeps the temporaries at a few (p1-p0)(q1-q0)
        g1 = normal_block(seed, TENSOR_IDS["B"], (L * n + p) * n + q)
        g2 = normal_block(seed, TENSOR_IDS["B"], (L * n + q) * n + p)
        res[L - L0] = (0.5 * math.exp(-L / (NL / 4.0))) * (g1 + g2)
    return res


def bvv_block(seed, o, v, NL, L0, L1, device, out=None):
    return bsym_block(seed, o + v, NL, L0, L1, o, o + v, o, o + v, device, out=out)


def make_inputs_device(o, v, NL, NP, NX, seed, device="cuda", with_bvv=True, z_scale=0.1):
    """dict of device tensors Xo, Xv, Z, B_ov, B_oo, B_vv (None if with_bvv=False), Y, V, eps  (recipe: generators.py)."""
    n = o + v
    dev = torch.device(device)
    eps_o = torch.sort(-1.5 + 1.2 * uniform_block(seed, TENSOR_IDS["eps_o"], torch.arange(o, device=dev))).values
    eps_v = torch.sort(0.1 + 2.9 * uniform_block(seed, TENSOR_IDS["eps_v"], torch.arange(v, device=dev))).values
    d = dict(eps=torch.cat([eps_o, eps_v]))
    d["Xo"] = _normal_full(seed, TENSOR_IDS["Xo"], (o, NP), dev) / math.sqrt(NP)
    d["Xv"] = _normal_full(seed, TENSOR_IDS["Xv"], (v, NP), dev) / math.sqrt(NP)
    G = _normal_full(seed, TENSOR_IDS["Z"], (NP, NP), dev)
    d["Z"] = (z_scale * 0.5) * (G + G.T)
    del G
    d["B_oo"] = bsym_block(seed, n, NL, 0, NL, 0, o, 0, o, dev)
    d["B_ov"] = bsym_block(seed, n, NL, 0, NL, 0, o, o, n, dev)
    d["B_vv"] = bvv_block(seed, o, v, NL, 0, NL, dev) if with_bvv else None
    d["Y"] = _normal_full(seed, TENSOR_IDS["Y"], (n, NX), dev) / math.sqrt(NX)
    G = _normal_full(seed, TENSOR_IDS["VG"], (NX, NX), dev)
    Vm = (G @ G.T) / NX            # input construction (a library GEMM), not part of the measured path
    d["V"] = 0.5 * (Vm + Vm.T)
    return d


def make_config_device(cfg: int, device="cuda", with_bvv=True):
    c = CONFIGS[cfg]
    return make_inputs_device(c["o"], c["v"], c["NL"], c["NP"], c["NX"], c["seed"], device=device, with_bvv=with_bvv)
