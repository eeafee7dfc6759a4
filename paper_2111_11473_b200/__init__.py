"""Thin Python binding of the C-ABI library `libthc_b200.so` (include/thc.h).

Argument marshalling only: every step of the residual/energy evaluation runs in the
library's own CUDA kernels.  torch is used for device memory and streams, nothing else.
There is no CPU path: importing works without a GPU (the CPU test-suite checks the
exported symbols), but every compute entry point raises if the library or a CUDA device
is missing.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libthc_b200.so")
SRC = os.path.join(_HERE, "csrc", "thc_lib.cu")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC"]

# every symbol include/thc.h declares
SYMBOLS = ("thc_setup", "thc_destroy", "thc_workspace_bytes", "thc_workspace_bytes_host", "thc_set_workspace",
           "thc_set_stream", "thc_get_blocks", "thc_residual", "thc_residual_terms", "thc_energy",
           "thc_energy_device", "thc_residual_host", "thc_profile_begin", "thc_profile_end", "thc_profile_work", "thc_kernel_launches", "thc_algorithmic_flops", "thc_dgemm",
           "thc_triple_product", "thc_strerror", "thc_last_cuda_error", "thc_last_error", "thc_shard_range",
           "thc_shard_doubles", "thc_residual_shard", "thc_residual_finish", "thc_energy_shard",
           "thc_profile_launches", "thc_profile_launch", "thc_algorithmic_work", "thc_probe", "thc_workspace_bytes_rr",
           "thc_residual_rr", "thc_workspace_bytes_t1", "thc_residual_t1", "thc_static_init", "thc_dgemm_static",
           "thc_workspace_bytes_mp2", "thc_mp2_density", "thc_workspace_bytes_als", "thc_cp_als_update")

STATIC_SCRATCH_BYTES = 16 << 20          # THC_STATIC_SCRATCH_BYTES of include/thc.h

TERM_NAMES = ("s1", "s2", "s3", "s6", "s7", "s9")
TERM_BITS = dict(s1=1, s2=2, s3=4, s6=8, s7=16, s9=32)


class ThcError(RuntimeError):
    pass


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile csrc/thc_lib.cu for sm_100a into libthc_b200.so (in-tree)."""
    deps = [os.path.join(_HERE, "csrc", f) for f in os.listdir(os.path.join(_HERE, "csrc"))]
    deps.append(os.path.join(os.path.dirname(_HERE), "include", "thc.h"))
    if (not force and os.path.exists(LIB_PATH)
            and all(os.path.getmtime(LIB_PATH) >= os.path.getmtime(d) for d in deps)):
        return LIB_PATH
    nvcc = os.environ.get("NVCC", "nvcc")
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB_PATH, SRC]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise ThcError("nvcc failed:\n" + r.stdout + r.stderr)
    if verbose:
        print(r.stderr)
    return LIB_PATH


class _Options(ctypes.Structure):
    _fields_ = [("bL", ctypes.c_int64), ("bP7", ctypes.c_int64), ("bX", ctypes.c_int64), ("bI", ctypes.c_int64),
                ("workspace_bytes_max", ctypes.c_int64), ("tma_min_flop", ctypes.c_int64), ("term_mask", ctypes.c_int32), ("device", ctypes.c_int32),
                ("bvv_mode", ctypes.c_int32), ("check_symmetry", ctypes.c_int32), ("use_graph", ctypes.c_int32),
                ("t2sq_algorithm", ctypes.c_int32)]


BVV_MODES = dict(device=0, host=1, provider=2)
_FILL_FN = ctypes.CFUNCTYPE(ctypes.c_int, ctypes.c_void_p, ctypes.c_int64, ctypes.c_int64, ctypes.c_void_p, ctypes.c_void_p)


class _BvvProvider(ctypes.Structure):
    _fields_ = [("fill", _FILL_FN), ("ctx", ctypes.c_void_p)]


class _DevView:
    """Zero-copy torch view of device memory the library owns (handed to a B_vv provider callback)."""

    def __init__(self, ptr, shape):
        self.__cuda_array_interface__ = dict(data=(int(ptr), False), shape=tuple(int(x) for x in shape), typestr="<f8",
                                             version=2, strides=None)


_lib = None


def lib() -> ctypes.CDLL:
    """Load the shared library (raises ThcError if it has not been built)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ThcError(f"{LIB_PATH} not found: run `python -c 'import __graft_entry__ as g; g.build()'` "
                       "(there is no fallback path)")
    L = ctypes.CDLL(LIB_PATH)
    P, D, I64, VP = ctypes.c_void_p, ctypes.c_double, ctypes.c_int64, ctypes.c_void_p
    L.thc_setup.argtypes = [ctypes.POINTER(VP), I64, I64, I64, I64, I64, ctypes.POINTER(_Options)]
    L.thc_destroy.argtypes = [VP]
    L.thc_workspace_bytes.argtypes = [VP]
    L.thc_workspace_bytes.restype = I64
    L.thc_workspace_bytes_host.argtypes = [VP]
    L.thc_workspace_bytes_host.restype = I64
    L.thc_set_workspace.argtypes = [VP, P, I64]
    L.thc_set_stream.argtypes = [VP, P]
    L.thc_get_blocks.argtypes = [VP, ctypes.POINTER(I64 * 4)]
    L.thc_residual.argtypes = [VP] + [P] * 10
    L.thc_residual_terms.argtypes = [VP] + [P] * 10 + [ctypes.POINTER(P * 6), P, P]
    L.thc_energy.argtypes = [VP, P, P, P, P, ctypes.POINTER(D)]
    L.thc_energy_device.argtypes = [VP, P, P, P, P, P]
    L.thc_profile_begin.argtypes = [VP, ctypes.c_int]
    L.thc_profile_end.argtypes = [VP, ctypes.POINTER(D * 3), ctypes.POINTER(I64 * 3)]
    L.thc_profile_work.argtypes = [VP, ctypes.POINTER(D * 3)]
    L.thc_profile_launches.argtypes = [VP]
    L.thc_profile_launches.restype = I64
    L.thc_profile_launch.argtypes = [VP, I64, ctypes.POINTER(ctypes.c_int), ctypes.POINTER(D), ctypes.POINTER(D),
                                     ctypes.c_char_p, I64]
    L.thc_algorithmic_work.argtypes = [VP, ctypes.POINTER(D * 3)]
    L.thc_last_error.argtypes = [VP]
    L.thc_probe.argtypes = [VP, ctypes.POINTER(D * 8)]
    L.thc_workspace_bytes_rr.argtypes = [VP, I64]
    L.thc_workspace_bytes_rr.restype = I64
    L.thc_residual_rr.argtypes = [VP, I64] + [P] * 12
    L.thc_workspace_bytes_t1.argtypes = [VP]
    L.thc_workspace_bytes_t1.restype = I64
    L.thc_residual_t1.argtypes = [VP] + [P] * 12 + [ctypes.POINTER(P * 6), ctypes.POINTER(P * 2), P, P]
    L.thc_residual_host.argtypes = [VP] + [P] * 10 + [ctypes.POINTER(D)]
    L.thc_kernel_launches.argtypes = [VP]
    L.thc_kernel_launches.restype = I64
    L.thc_algorithmic_flops.argtypes = [VP]
    L.thc_algorithmic_flops.restype = D
    L.thc_dgemm.argtypes = [VP, ctypes.c_int, ctypes.c_int, I64, I64, I64, D, P, I64, P, I64, D, P, I64]
    L.thc_triple_product.argtypes = [VP, I64, I64, I64, P, P, P, P, ctypes.c_int]
    L.thc_shard_range.argtypes = [I64, I64, ctypes.c_int, ctypes.c_int, ctypes.POINTER(I64 * 4)]
    L.thc_shard_doubles.argtypes = [VP]
    L.thc_shard_doubles.restype = I64
    L.thc_residual_shard.argtypes = [VP] + [P] * 9 + [ctypes.c_int, ctypes.c_int, P]
    L.thc_residual_finish.argtypes = [VP] + [P] * 6 + [P, P, ctypes.POINTER(P * 6)]
    L.thc_energy_shard.argtypes = [VP, P, P, P, P, ctypes.c_int, ctypes.c_int, P]
    L.thc_strerror.argtypes = [ctypes.c_int]
    L.thc_strerror.restype = ctypes.c_char_p
    L.thc_last_cuda_error.argtypes = [VP]
    L.thc_static_init.argtypes = [ctypes.c_int]
    L.thc_workspace_bytes_mp2.argtypes = [VP]
    L.thc_workspace_bytes_mp2.restype = I64
    L.thc_mp2_density.argtypes = [VP, P, P, P, P, P]
    L.thc_workspace_bytes_als.argtypes = [VP, I64, I64, I64, I64]
    L.thc_workspace_bytes_als.restype = I64
    L.thc_cp_als_update.argtypes = [VP, I64, I64, I64, I64, P, P, P, P, ctypes.c_int, P]
    L.thc_dgemm_static.argtypes = [ctypes.c_int, P, I64, I64, I64, ctypes.c_int, D, P, I64, P, I64, D, P, I64]
    for name in SYMBOLS:
        getattr(L, name)          # AttributeError if a declared symbol is missing
    _lib = L
    return L


def _check(st: int, h=None):
    if st != 0:
        msg = lib().thc_strerror(st).decode()
        if h is not None and st == -4:
            msg += f" [cudaError {lib().thc_last_error(h)}]"
        raise ThcError(f"thc status {st}: {msg}")


def thc_static_init(device: int = -1):
    """Once-per-device set-up of the allocation-free entry point (include/thc.h)."""
    _check(lib().thc_static_init(int(device)))


def thc_dgemm_static(A, B, C, alpha: float = 1.0, beta: float = 0.0, splits: int = 0):
    """C[M][N] = alpha * A[M][K] B[N][K]^T + beta * C through thc_dgemm_static (include/thc.h): no handle, no workspace, no
    cudaMalloc; split-K partials in the library's static device array (STATIC_SCRATCH_BYTES).  Runs on torch's current
    stream of the tensors' device.  Argument marshalling only."""
    import torch
    for name, t in (("A", A), ("B", B), ("C", C)):
        if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != torch.float64 or t.dim() != 2 or t.stride(1) != 1:
            raise ThcError(f"{name}: need a 2-D float64 CUDA tensor with unit inner stride")
    M, K = A.shape
    N = B.shape[0]
    if B.shape[1] != K or tuple(C.shape) != (M, N) or A.device != B.device or A.device != C.device:
        raise ThcError("thc_dgemm_static: shapes / devices do not match")
    dev = A.device.index
    stream = torch.cuda.current_stream(A.device).cuda_stream
    _check(lib().thc_dgemm_static(dev, ctypes.c_void_p(stream), M, N, K, int(splits), float(alpha),
                                  ctypes.c_void_p(A.data_ptr()), A.stride(0), ctypes.c_void_p(B.data_ptr()), B.stride(0),
                                  float(beta), ctypes.c_void_p(C.data_ptr()), C.stride(0)))


def _dev_ptr(t, name, numel=None):
    import torch
    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous():
        raise ThcError(f"{name}: need a contiguous float64 CUDA tensor")
    if numel is not None and t.numel() != numel:
        raise ThcError(f"{name}: expected {numel} elements, got {t.numel()}")
    return ctypes.c_void_p(t.data_ptr())


def _host_ptr(t, name, numel):
    import torch
    if not isinstance(t, torch.Tensor) or t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous():
        raise ThcError(f"{name}: need a contiguous float64 CPU tensor")
    if t.numel() != numel:
        raise ThcError(f"{name}: expected {numel} elements, got {t.numel()}")
    return ctypes.c_void_p(t.data_ptr())


class Thc:
    """One problem shape (thc_setup ... thc_destroy).  Methods mirror the C entry points."""

    def __init__(self, o, v, NL, NP, NX, *, bL=0, bP7=0, bX=0, bI=0, workspace_bytes_max=0, term_mask=0,
                 device=-1, torch_workspace=True, bvv_mode="device", check_symmetry=False, use_graph=-1, tma_min_flop=0,
                 t2sq_algorithm=0):
        import torch
        if not torch.cuda.is_available():
            raise ThcError("no CUDA device: the THC residual has no CPU path")
        self.o, self.v, self.NL, self.NP, self.NX = o, v, NL, NP, NX
        self._h = ctypes.c_void_p()
        self.bvv_mode = bvv_mode
        opt = _Options(bL, bP7, bX, bI, workspace_bytes_max, tma_min_flop, term_mask, device, BVV_MODES[bvv_mode],
                       int(bool(check_symmetry)), int(use_graph), int(t2sq_algorithm))
        _check(lib().thc_setup(ctypes.byref(self._h), o, v, NL, NP, NX, ctypes.byref(opt)))
        self._ws = None
        self._torch_ws = torch_workspace
        self._device = torch.device("cuda", torch.cuda.current_device() if device < 0 else device)

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value and _lib is not None:
            _lib.thc_destroy(self._h)
            self._h = ctypes.c_void_p()
            self._ws = None

    __del__ = close

    # ---- plumbing -----------------------------------------------------------------------------------------
    def _prepare(self, nbytes):
        """Workspace from torch's allocator, work on torch's current stream."""
        import torch
        if self._torch_ws and (self._ws is None or self._ws.numel() < nbytes):
            self._ws = None
            self._ws = torch.empty(nbytes, dtype=torch.uint8, device=self._device)
            _check(lib().thc_set_workspace(self._h, ctypes.c_void_p(self._ws.data_ptr()), self._ws.numel()), self._h)
        _check(lib().thc_set_stream(self._h, ctypes.c_void_p(torch.cuda.current_stream(self._device).cuda_stream)))

    @property
    def workspace_bytes(self):
        return int(lib().thc_workspace_bytes(self._h))

    @property
    def workspace_bytes_host(self):
        return int(lib().thc_workspace_bytes_host(self._h))

    @property
    def blocks(self):
        out = (ctypes.c_int64 * 4)()
        _check(lib().thc_get_blocks(self._h, ctypes.byref(out)))
        return dict(bL=out[0], bP7=out[1], bX=out[2], bI=out[3])

    @property
    def kernel_launches(self):
        return int(lib().thc_kernel_launches(self._h))

    @property
    def algorithmic_flops(self):
        return float(lib().thc_algorithmic_flops(self._h))

    def _bvv_ptr(self, B_vv, conv):
        """B_vv argument per thc_bvv_mode: device tensor, host tensor, or a callable fill(L0, nl, dst) that writes
        B_vv[L0:L0+nl] into the device tensor dst[nl, v, v] on torch's current stream."""
        import torch
        v, NL = self.v, self.NL
        if self.bvv_mode == "device":
            return conv(B_vv, "B_vv", NL * v * v)
        if self.bvv_mode == "host":
            return _host_ptr(B_vv, "B_vv", NL * v * v)
        if not callable(B_vv):
            raise ThcError("B_vv: bvv_mode='provider' needs a callable fill(L0, nl, dst)")

        def _fill(ctx, L0, nl, dst, stream):
            try:
                # ExternalStream(0) would hand out a NEW pool stream, not the legacy default stream the library is on
                lib_stream = (torch.cuda.ExternalStream(stream, device=self._device) if stream
                              else torch.cuda.default_stream(self._device))
                with torch.cuda.stream(lib_stream):
                    B_vv(int(L0), int(nl), torch.as_tensor(_DevView(dst, (nl, v, v)), device=self._device))
                return 0
            except Exception as exc:            # never let an exception cross the C ABI
                self._provider_error = exc
                return 1

        self._provider = _BvvProvider(_FILL_FN(_fill), None)     # kept alive for the duration of the call
        return ctypes.cast(ctypes.pointer(self._provider), ctypes.c_void_p)

    def _in_ptrs(self, Xo, Xv, Z, B_ov, B_oo, B_vv, Y, V, eps, conv):
        o, v, NL, NP, NX = self.o, self.v, self.NL, self.NP, self.NX
        return [conv(Xo, "Xo", o * NP), conv(Xv, "Xv", v * NP), conv(Z, "Z", NP * NP),
                conv(B_ov, "B_ov", NL * o * v), conv(B_oo, "B_oo", NL * o * o), self._bvv_ptr(B_vv, conv),
                conv(Y, "Y", (o + v) * NX), conv(V, "V", NX * NX), conv(eps, "eps", o + v)]

    # ---- entry points ---------------------------------------------------------------------------------------
    def thc_residual(self, Xo, Xv, Z, B_ov, B_oo, B_vv, Y, V, eps, out=None):
        """R_PQ [NP, NP] (device tensor; asynchronous on torch's current stream)."""
        import torch
        self._prepare(self.workspace_bytes)
        R = out if out is not None else torch.empty(self.NP, self.NP, dtype=torch.float64, device=self._device)
        ptrs = self._in_ptrs(Xo, Xv, Z, B_ov, B_oo, B_vv, Y, V, eps, _dev_ptr)
        _check(lib().thc_residual(self._h, *ptrs, _dev_ptr(R, "R", self.NP * self.NP)), self._h)
        return R

    def thc_residual_terms(self, Xo, Xv, Z, B_ov, B_oo, B_vv, Y, V, eps):
        """dict with R, s1, s2, s3, s6, s7, s9 [NP, NP], xi_oo [o, o], xi_vv [v, v] (device tensors)."""
        import torch
        self._prepare(self.workspace_bytes)
        kw = dict(dtype=torch.float64, device=self._device)
        res = {k: torch.empty(self.NP, self.NP, **kw) for k in ("R",) + TERM_NAMES}
        res["xi_oo"] = torch.empty(self.o, self.o, **kw)
        res["xi_vv"] = torch.empty(self.v, self.v, **kw)
        terms = (ctypes.c_void_p * 6)(*[res[k].data_ptr() for k in TERM_NAMES])
        ptrs = self._in_ptrs(Xo, Xv, Z, B_ov, B_oo, B_vv, Y, V, eps, _dev_ptr)
        _check(lib().thc_residual_terms(self._h, *ptrs, _dev_ptr(res["R"], "R"), ctypes.byref(terms),
                                        _dev_ptr(res["xi_oo"], "xi_oo"), _dev_ptr(res["xi_vv"], "xi_vv")), self._h)
        return res

    def thc_residual_t1(self, Xo, Xv, Z, t1, B_ov, B_oo, B_vv, Y, V, eps):
        """T1-dressed evaluation: dict with R, s1..s9 [NP, NP], sigma, sigma_GH, sigma_IJ [o, v], xi_oo, xi_vv."""
        import torch
        self._prepare(max(self.workspace_bytes, int(lib().thc_workspace_bytes_t1(self._h))))
        kw = dict(dtype=torch.float64, device=self._device)
        res = {k: torch.empty(self.NP, self.NP, **kw) for k in ("R",) + TERM_NAMES}
        for k in ("sigma", "sigma_GH", "sigma_IJ"):
            res[k] = torch.empty(self.o, self.v, **kw)
        res["xi_oo"], res["xi_vv"] = torch.empty(self.o, self.o, **kw), torch.empty(self.v, self.v, **kw)
        terms = (ctypes.c_void_p * 6)(*[res[k].data_ptr() for k in TERM_NAMES])
        parts = (ctypes.c_void_p * 2)(res["sigma_GH"].data_ptr(), res["sigma_IJ"].data_ptr())
        p = self._in_ptrs(Xo, Xv, Z, B_ov, B_oo, B_vv, Y, V, eps, _dev_ptr)
        _check(lib().thc_residual_t1(self._h, p[0], p[1], p[2], _dev_ptr(t1, "t1", self.o * self.v), p[3], p[4], p[5], p[6],
                                     p[7], p[8], _dev_ptr(res["R"], "R"), _dev_ptr(res["sigma"], "sigma"), ctypes.byref(terms),
                                     ctypes.byref(parts), _dev_ptr(res["xi_oo"], "xi_oo"), _dev_ptr(res["xi_vv"], "xi_vv")), self._h)
        return res

    def thc_residual_rr(self, tau, T, Xo, Xv, B_ov, B_oo, B_vv, Y, V, eps, want_Z=False):
        """R_rr [NR, NR] = tau R(Z) tau^T with Z = tau^T T tau (rank-reduced working variables; device tensors)."""
        import torch
        NR = int(tau.shape[0])
        o, v, NL, NP, NX = self.o, self.v, self.NL, self.NP, self.NX
        self._prepare(int(lib().thc_workspace_bytes_rr(self._h, NR)))
        kw = dict(dtype=torch.float64, device=self._device)
        R_rr = torch.empty(NR, NR, **kw)
        Z = torch.empty(NP, NP, **kw) if want_Z else None
        _check(lib().thc_residual_rr(
            self._h, NR, _dev_ptr(tau, "tau", NR * NP), _dev_ptr(T, "T", NR * NR), _dev_ptr(Xo, "Xo", o * NP),
            _dev_ptr(Xv, "Xv", v * NP), _dev_ptr(B_ov, "B_ov", NL * o * v), _dev_ptr(B_oo, "B_oo", NL * o * o),
            self._bvv_ptr(B_vv, _dev_ptr), _dev_ptr(Y, "Y", (o + v) * NX), _dev_ptr(V, "V", NX * NX),
            _dev_ptr(eps, "eps", o + v), _dev_ptr(R_rr, "R_rr"), _dev_ptr(Z, "Z") if want_Z else None), self._h)
        return (R_rr, Z) if want_Z else R_rr

    def thc_energy(self, Xo, Xv, Z, B_ov) -> float:
        self._prepare(self.workspace_bytes)
        o, v, NL, NP = self.o, self.v, self.NL, self.NP
        E = ctypes.c_double(0.0)
        _check(lib().thc_energy(self._h, _dev_ptr(Xo, "Xo", o * NP), _dev_ptr(Xv, "Xv", v * NP),
                                _dev_ptr(Z, "Z", NP * NP), _dev_ptr(B_ov, "B_ov", NL * o * v), ctypes.byref(E)), self._h)
        return E.value

    def thc_energy_device(self, Xo, Xv, Z, B_ov, out=None):
        """E as a 1-element device tensor (asynchronous on torch's current stream)."""
        import torch
        self._prepare(self.workspace_bytes)
        o, v, NL, NP = self.o, self.v, self.NL, self.NP
        E = out if out is not None else torch.empty(1, dtype=torch.float64, device=self._device)
        _check(lib().thc_energy_device(self._h, _dev_ptr(Xo, "Xo", o * NP), _dev_ptr(Xv, "Xv", v * NP),
                                       _dev_ptr(Z, "Z", NP * NP), _dev_ptr(B_ov, "B_ov", NL * o * v),
                                       _dev_ptr(E, "E", 1)), self._h)
        return E

    # ---- sharded evaluation (one handle per device; the caller sums `packed` over the ranks) -------------------------
    @property
    def shard_doubles(self):
        return int(lib().thc_shard_doubles(self._h))

    def _slice_ptr(self, t, name, numel):
        return ctypes.c_void_p(None) if numel == 0 else _dev_ptr(t, name, numel)

    def thc_residual_shard(self, Xo, Xv, Z, B_ov, B_oo, B_vv, Y, V, eps, rank, nranks, out=None):
        """This rank's packed partial sums (device tensor of shard_doubles); B_* are the rank's own L-slices."""
        import torch
        self._prepare(self.workspace_bytes)
        o, v, NP, NX = self.o, self.v, self.NP, self.NX
        L0, L1, _, _ = thc_shard_range(self.NL, NP, rank, nranks)
        nl = L1 - L0
        packed = out if out is not None else torch.empty(self.shard_doubles, dtype=torch.float64, device=self._device)
        if self.bvv_mode == "device":
            bvv = self._slice_ptr(B_vv, "B_vv", nl * v * v)
        elif self.bvv_mode == "host":
            # the C entry expects the rank's own slice (vector L_begin first); the whole host array is accepted too
            import torch
            if isinstance(B_vv, torch.Tensor) and B_vv.numel() == self.NL * v * v and nl != self.NL:
                B_vv = B_vv.reshape(self.NL, v, v)[L0:L1]
            bvv = ctypes.c_void_p(None) if nl == 0 else _host_ptr(B_vv, "B_vv", nl * v * v)
        else:
            bvv = self._bvv_ptr(B_vv, _dev_ptr)      # provider: fill() receives global Cholesky indices
        _check(lib().thc_residual_shard(
            self._h, _dev_ptr(Xo, "Xo", o * NP), _dev_ptr(Xv, "Xv", v * NP), _dev_ptr(Z, "Z", NP * NP),
            self._slice_ptr(B_ov, "B_ov", nl * o * v), self._slice_ptr(B_oo, "B_oo", nl * o * o), bvv,
            _dev_ptr(Y, "Y", (o + v) * NX), _dev_ptr(V, "V", NX * NX), _dev_ptr(eps, "eps", o + v), rank, nranks,
            _dev_ptr(packed, "packed", self.shard_doubles)), self._h)
        return packed

    def thc_residual_finish(self, Xo, Xv, Z, Y, V, eps, packed, want_terms=False):
        """R (and optionally every term) from the rank-summed packed buffer, which is modified."""
        import torch
        self._prepare(self.workspace_bytes)
        o, v, NP, NX = self.o, self.v, self.NP, self.NX
        kw = dict(dtype=torch.float64, device=self._device)
        res = {"R": torch.empty(NP, NP, **kw)}
        terms = None
        if want_terms:
            for k in TERM_NAMES:
                res[k] = torch.empty(NP, NP, **kw)
            terms = ctypes.byref((ctypes.c_void_p * 6)(*[res[k].data_ptr() for k in TERM_NAMES]))
        _check(lib().thc_residual_finish(
            self._h, _dev_ptr(Xo, "Xo", o * NP), _dev_ptr(Xv, "Xv", v * NP), _dev_ptr(Z, "Z", NP * NP),
            _dev_ptr(Y, "Y", (o + v) * NX), _dev_ptr(V, "V", NX * NX), _dev_ptr(eps, "eps", o + v),
            _dev_ptr(packed, "packed", self.shard_doubles), _dev_ptr(res["R"], "R"), terms), self._h)
        return res if want_terms else res["R"]

    def thc_energy_shard(self, Xo, Xv, Z, B_ov, rank, nranks, out=None):
        import torch
        self._prepare(self.workspace_bytes)
        o, v, NP = self.o, self.v, self.NP
        L0, L1, _, _ = thc_shard_range(self.NL, NP, rank, nranks)
        E = out if out is not None else torch.empty(1, dtype=torch.float64, device=self._device)
        _check(lib().thc_energy_shard(self._h, _dev_ptr(Xo, "Xo", o * NP), _dev_ptr(Xv, "Xv", v * NP),
                                      _dev_ptr(Z, "Z", NP * NP), self._slice_ptr(B_ov, "B_ov", (L1 - L0) * o * v),
                                      rank, nranks, _dev_ptr(E, "E", 1)), self._h)
        return E

    def thc_profile_begin(self, class_mask=7):
        _check(lib().thc_profile_begin(self._h, int(class_mask)), self._h)

    def thc_profile_end(self):
        """{class: (milliseconds, launches)} for classes gemm / triple / ew; synchronises the stream."""
        ms, cnt = (ctypes.c_double * 3)(), (ctypes.c_int64 * 3)()
        _check(lib().thc_profile_end(self._h, ctypes.byref(ms), ctypes.byref(cnt)), self._h)
        return {k: (ms[i], cnt[i]) for i, k in enumerate(("gemm", "triple", "ew"))}

    def thc_profile_work(self):
        """{class: executed flop (gemm, triple) or algorithmic HBM bytes (ew)} of the last thc_profile_end."""
        w = (ctypes.c_double * 3)()
        _check(lib().thc_profile_work(self._h, ctypes.byref(w)), self._h)
        return {k: w[i] for i, k in enumerate(("gemm", "triple", "ew"))}

    def thc_profile_launches(self):
        """[(class name, milliseconds, work, description)] of every launch timed by the last thc_profile_end."""
        n = int(lib().thc_profile_launches(self._h))
        out, names = [], ("gemm", "triple", "ew")
        buf = ctypes.create_string_buffer(192)
        for k in range(n):
            cls, ms, work = ctypes.c_int(), ctypes.c_double(), ctypes.c_double()
            _check(lib().thc_profile_launch(self._h, k, ctypes.byref(cls), ctypes.byref(ms), ctypes.byref(work), buf,
                                            len(buf)), self._h)
            out.append((names[cls.value], ms.value, work.value, buf.value.decode()))
        return out

    @property
    def algorithmic_work(self):
        """{class: algorithmic flop of one evaluation}: gemm (every GEMM-shaped step), triple (Alg.6 line 11), ew (H3)."""
        w = (ctypes.c_double * 3)()
        _check(lib().thc_algorithmic_work(self._h, ctypes.byref(w)), self._h)
        return {k: w[i] for i, k in enumerate(("gemm", "triple", "ew"))}

    def thc_probe(self):
        """Measured ceilings of the device (thc.h): FP64 tensor / FMA issue rates, shared-memory load bandwidth."""
        out = (ctypes.c_double * 8)()
        _check(lib().thc_probe(self._h, ctypes.byref(out)), self._h)
        return dict(dmma_tflops=out[0], dfma_tflops=out[1], dmma_plus_dfma_interleaved_tflops=out[2],
                    lds32_bytes_per_clk_per_sm=out[3], lds64_bytes_per_clk_per_sm=out[4],
                    lds128_bytes_per_clk_per_sm=out[5], sm_clock_mhz=out[6])

    def thc_residual_host(self, Xo, Xv, Z, B_ov, B_oo, B_vv, Y, V, eps, R_host, want_energy=True):
        """End-to-end entry: HOST tensors in, R written into the host tensor R_host, returns E (or None)."""
        self._prepare(self.workspace_bytes_host)
        ptrs = self._in_ptrs(Xo, Xv, Z, B_ov, B_oo, B_vv, Y, V, eps, _host_ptr)
        E = ctypes.c_double(0.0)
        _check(lib().thc_residual_host(self._h, *ptrs, _host_ptr(R_host, "R_host", self.NP * self.NP),
                                       ctypes.byref(E) if want_energy else None), self._h)
        return E.value if want_energy else None

    def thc_mp2_density(self, Xo, Xv, Z):
        """(D_oo [o, o], D_vv [v, v]) of PAPER.md Eqs.47-48 (App.II) for the THC amplitudes (Xo, Xv, Z)."""
        import torch
        need = lib().thc_workspace_bytes_mp2(self._h)
        if need < 0:
            _check(int(need), self._h)
        self._prepare(max(self.workspace_bytes, need))
        D_oo = torch.empty(self.o, self.o, dtype=torch.float64, device=self._device)
        D_vv = torch.empty(self.v, self.v, dtype=torch.float64, device=self._device)
        _check(lib().thc_mp2_density(self._h, _dev_ptr(Xo, "Xo", self.o * self.NP), _dev_ptr(Xv, "Xv", self.v * self.NP),
                                     _dev_ptr(Z, "Z", self.NP * self.NP), _dev_ptr(D_oo, "D_oo"), _dev_ptr(D_vv, "D_vv")), self._h)
        return D_oo, D_vv

    def thc_cp_als_update(self, A, Y, Z, X, iters, want_rnorm2=False):
        """One ALS update of the factor X [I, N] in place (App.I, Eqs.44-46; `iters` PCG iterations from X)."""
        import torch
        I, J, K = A.shape
        N = X.shape[1]
        need = lib().thc_workspace_bytes_als(self._h, I, J, K, N)
        if need < 0:
            _check(int(need), self._h)
        self._prepare(max(self.workspace_bytes, need))
        rn = torch.empty(I, dtype=torch.float64, device=self._device) if want_rnorm2 else None
        _check(lib().thc_cp_als_update(self._h, I, J, K, N, _dev_ptr(A, "A", I * J * K), _dev_ptr(Y, "Y", J * N),
                                       _dev_ptr(Z, "Z", K * N), _dev_ptr(X, "X", I * N), int(iters),
                                       _dev_ptr(rn, "rnorm2") if want_rnorm2 else None), self._h)
        return rn

    def thc_dgemm(self, a_kmajor, b_kmajor, M, N, K, alpha, A, lda, B, ldb, beta, C, ldc):
        # room for the split-K partial tiles of a skinny product (at most 64 splits of < 148 tiles)
        self._prepare(self.workspace_bytes + 8 * 64 * min(M * N, 148 * 128 * 128) + 4096)
        _check(lib().thc_dgemm(self._h, int(a_kmajor), int(b_kmajor), M, N, K, alpha, _dev_ptr(A, "A"), lda,
                               _dev_ptr(B, "B"), ldb, beta, _dev_ptr(C, "C"), ldc), self._h)

    def thc_triple_product(self, nI, nPp, NPp, E, F, G, H, accumulate):
        self._prepare(self.workspace_bytes)
        _check(lib().thc_triple_product(self._h, nI, nPp, NPp, _dev_ptr(E, "E", nI * nPp * NPp),
                                        _dev_ptr(F, "F", nI * nPp * NPp), _dev_ptr(G, "G", nI * NPp * NPp),
                                        _dev_ptr(H, "H", nPp * NPp * NPp), int(accumulate)), self._h)


def thc_shard_range(NL, NP, rank, nranks):
    """(L_begin, L_end, P_begin, P_end) of one rank: its Cholesky range and its row block of the T2^2 terms."""
    out = (ctypes.c_int64 * 4)()
    _check(lib().thc_shard_range(NL, NP, rank, nranks, ctypes.byref(out)))
    return tuple(int(x) for x in out)


def thc_setup(o, v, NL, NP, NX, **options) -> Thc:
    return Thc(o, v, NL, NP, NX, **options)
