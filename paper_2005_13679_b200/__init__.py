"""paper_2005_13679_b200 -- thin Python binding of libmcb (include/mcb.h).

Argument marshalling only: every step of the hot path (Algorithm 1 / 2 batches, hashing table, jump maps,
H.C) runs in the hand-written sm_100a kernels behind the C ABI.  PyTorch is used for device memory and
streams.  There is no CPU fallback: importing works without a GPU (so the symbol table can be checked), but
any compute call without the built library or without a CUDA device raises.

Names follow include/mcb.h: Space.unrank / rank / build_structure / hc_apply / hc_apply_host ...
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmcb.so")

OK, EINVAL, ERANGE, ENOMEM, ECUDA, ENOTREADY, EUNSUPPORTED, ESCRATCH = 0, -1, -2, -3, -4, -5, -6, -7
TRUNCATED = 1          # mcb_lanczos only: completed with fewer steps than the paper's nc / 8
FOCK_TABLE, MAP1, MAP2, MAP2C = 0, 1, 2, 3
AUTO, MAPS, REHASH, GEMM, RUNS, SPARSE = 0, 1, 2, 3, 4, 5
MAX_M, MAX_M_APPLY, MAX_M_TILED = 32, 32, 12
RHO_STATIC_MAX_M, RHO_STATIC_BYTES = 12, 8 << 20

EXPORTS = (
    "mcb_space_create", "mcb_space_destroy", "mcb_nc", "mcb_nc_removed", "mcb_binom_table",
    "mcb_unrank", "mcb_rank", "mcb_structure_bytes", "mcb_build_structure", "mcb_detach_structure",
    "mcb_fock_export", "mcb_map1_export", "mcb_map2_export", "mcb_map2c_export", "mcb_apply_workspace_bytes",
    "mcb_hc_apply", "mcb_hc_apply_host", "mcb_last_apply_launches", "mcb_timing_enable", "mcb_timing_read", "mcb_fp64_peak", "mcb_strerror", "mcb_last_cuda_error",
    "mcb_rho_workspace_bytes", "mcb_rho", "mcb_lanczos_workspace_bytes", "mcb_lanczos", "mcb_resolve_mode",
    "mcb_lanczos_steps", "mcb_tridiag_eigvals", "mcb_debug_bounds", "mcb_rho_static", "mcb_last_apply_memops",
)

_lib = None


class McbError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        msg = lib().mcb_strerror(status).decode()
        if status == ECUDA:
            msg += f" [cudaError {lib().mcb_last_cuda_error()}]"
        super().__init__(f"{where}: {msg} ({status})")


def lib():
    """Load libmcb.so (built in-tree by paper_2005_13679_b200.build); fails loudly if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2005_13679_b200.build` "
                              "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        vp, ll, i = ctypes.c_void_p, ctypes.c_longlong, ctypes.c_int
        L.mcb_space_create.argtypes = [i, i, ctypes.POINTER(vp)]
        L.mcb_space_destroy.argtypes = [vp]
        L.mcb_space_destroy.restype = None
        L.mcb_nc.argtypes = [vp]; L.mcb_nc.restype = ll
        L.mcb_nc_removed.argtypes = [vp, i]; L.mcb_nc_removed.restype = ll
        L.mcb_binom_table.argtypes = [vp, vp]
        L.mcb_unrank.argtypes = [vp, vp, ll, vp, vp]
        L.mcb_rank.argtypes = [vp, vp, ll, vp, vp]
        L.mcb_structure_bytes.argtypes = [vp, i]; L.mcb_structure_bytes.restype = ll
        L.mcb_build_structure.argtypes = [vp, i, vp, ll, vp]
        L.mcb_detach_structure.argtypes = [vp, i]
        L.mcb_fock_export.argtypes = [vp, i, ll, ll, vp]
        L.mcb_map1_export.argtypes = [vp, ll, ll, vp]
        L.mcb_map2_export.argtypes = [vp, ll, ll, vp]
        L.mcb_map2c_export.argtypes = [vp, ll, ll, vp, vp, ll]
        L.mcb_apply_workspace_bytes.argtypes = [vp, i]; L.mcb_apply_workspace_bytes.restype = ll
        L.mcb_hc_apply.argtypes = [vp, vp, vp, vp, vp, i, vp, vp]
        L.mcb_hc_apply_host.argtypes = [vp, vp, vp, vp, vp, i, vp, vp, vp, vp]
        L.mcb_last_apply_launches.argtypes = [vp]
        L.mcb_last_apply_memops.argtypes = [vp, ctypes.POINTER(i), ctypes.POINTER(i)]
        L.mcb_timing_enable.argtypes = [vp, i]
        L.mcb_timing_read.argtypes = [vp, i, vp, vp]
        L.mcb_fp64_peak.argtypes = [i, ctypes.POINTER(ctypes.c_double), vp]
        L.mcb_resolve_mode.argtypes = [vp, vp, vp, i]
        L.mcb_rho_workspace_bytes.argtypes = [vp]; L.mcb_rho_workspace_bytes.restype = ll
        L.mcb_rho.argtypes = [vp, vp, vp, vp, vp, vp]
        L.mcb_rho_static.argtypes = [vp, vp, vp, vp, vp]
        L.mcb_lanczos_workspace_bytes.argtypes = [vp, i]; L.mcb_lanczos_workspace_bytes.restype = ll
        L.mcb_lanczos.argtypes = [vp, vp, vp, vp, i, i, ctypes.c_double, vp, vp, ctypes.POINTER(i), vp, vp, vp]
        L.mcb_debug_bounds.argtypes = [vp, vp]
        L.mcb_lanczos_steps.argtypes = [vp, i]
        L.mcb_tridiag_eigvals.argtypes = [i, vp, vp, vp]
        L.mcb_strerror.argtypes = [i]; L.mcb_strerror.restype = ctypes.c_char_p
        L.mcb_last_cuda_error.argtypes = []
        _lib = L
    return _lib


def _check(status: int, where: str):
    if status != OK:
        raise McbError(status, where)


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_2005_13679_b200 needs a CUDA device (no CPU fallback)")
    return torch


def _stream_ptr(stream) -> int:
    torch = _torch()
    s = stream if stream is not None else torch.cuda.current_stream()
    return int(s.cuda_stream)


def _host_c128(a, shape) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.complex128)
    if a.size != int(np.prod(shape)):
        raise ValueError(f"expected {shape} complex values, got {a.shape}")
    return a


def fp64_peak(kind: int = 0, stream=None) -> float:
    """Measured FP64 TFLOP/s of the current device: kind 0 DFMA, 1 DMMA m8n8k4, 2 both interleaved."""
    out = ctypes.c_double(0.0)
    _check(lib().mcb_fp64_peak(kind, ctypes.byref(out), _stream_ptr(stream)), "mcb_fp64_peak")
    return float(out.value)


def tridiag_eigvals(alpha, beta) -> np.ndarray:
    """Ascending eigenvalues of the real symmetric tridiagonal matrix with diagonal alpha[0..n-1] and off-diagonal
    beta[0..n-2] (mcb_tridiag_eigvals: the host-side finish of the Lanczos run).  Host only."""
    a = np.ascontiguousarray(alpha, dtype=np.float64)
    n = int(a.size)
    b = np.ascontiguousarray(np.asarray(beta, dtype=np.float64)[:max(n - 1, 0)])
    if n > 1 and b.size < n - 1:
        raise ValueError("beta needs at least n - 1 entries")
    out = np.empty(n, dtype=np.float64)
    bb = b if b.size else np.zeros(1)
    _check(lib().mcb_tridiag_eigvals(n, a.ctypes.data, bb.ctypes.data, out.ctypes.data), "mcb_tridiag_eigvals")
    return out


class Space:
    """N bosons in M orbitals (include/mcb.h mcb_space).  Owns the torch buffers of the structures it builds."""

    def __init__(self, N: int, M: int, device=None):
        torch = _torch()
        self.N, self.M = int(N), int(M)
        self.P = self.M * (self.M + 1) // 2
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        self._h = ctypes.c_void_p()
        with torch.cuda.device(self.device):
            _check(lib().mcb_space_create(self.N, self.M, ctypes.byref(self._h)), "mcb_space_create")
        self.nc = int(lib().mcb_nc(self._h))
        self.nc2 = int(lib().mcb_nc_removed(self._h, 2))
        self._buffers = {}
        self._workspace = {}

    # -- lifetime -----------------------------------------------------------------------------------------
    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            _torch().cuda.synchronize(self.device)
            lib().mcb_space_destroy(self._h)
            self._h = ctypes.c_void_p()
            self._buffers.clear()
            self._workspace.clear()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- tables -------------------------------------------------------------------------------------------
    def binom_table(self) -> np.ndarray:
        out = np.zeros((self.N + 1, self.M + 1), dtype=np.int64)
        _check(lib().mcb_binom_table(self._h, out.ctypes.data), "mcb_binom_table")
        return out

    def nc_removed(self, r: int) -> int:
        return int(lib().mcb_nc_removed(self._h, r))

    # -- batched hashing ------------------------------------------------------------------------------------
    def unrank(self, idx, stream=None):
        """int32 device tensor [batch] -> int32 device tensor [batch, M] (Algorithm 2)."""
        torch = _torch()
        idx = idx.to(device=self.device, dtype=torch.int32).contiguous()
        occ = torch.empty((idx.numel(), self.M), dtype=torch.int32, device=self.device)
        with torch.cuda.device(self.device):
            _check(lib().mcb_unrank(self._h, idx.data_ptr(), idx.numel(), occ.data_ptr(), _stream_ptr(stream)), "mcb_unrank")
        return occ

    def rank(self, occ, stream=None):
        """int32 device tensor [batch, M] -> int32 device tensor [batch] (Algorithm 1)."""
        torch = _torch()
        occ = occ.to(device=self.device, dtype=torch.int32).contiguous().view(-1, self.M)
        idx = torch.empty((occ.shape[0],), dtype=torch.int32, device=self.device)
        with torch.cuda.device(self.device):
            _check(lib().mcb_rank(self._h, occ.data_ptr(), occ.shape[0], idx.data_ptr(), _stream_ptr(stream)), "mcb_rank")
        return idx

    # -- structures ---------------------------------------------------------------------------------------
    def structure_bytes(self, which: int) -> int:
        n = int(lib().mcb_structure_bytes(self._h, which))
        if n < 0:
            raise McbError(n, "mcb_structure_bytes")
        return n

    def build_structure(self, which: int, stream=None, buf=None):
        """Build the structure into a torch buffer of mcb_structure_bytes (allocated here unless `buf`, a uint8 CUDA tensor
        of at least that size, is given -- e.g. to rebuild in place)."""
        torch = _torch()
        nbytes = self.structure_bytes(which)
        if buf is None:
            buf = torch.empty(max(nbytes, 256), dtype=torch.uint8, device=self.device)
        elif buf.dtype != torch.uint8 or not buf.is_cuda or buf.device != self.device or buf.numel() < nbytes or not buf.is_contiguous():
            raise ValueError("buf must be a contiguous uint8 CUDA tensor of at least structure_bytes on the space's device")
        assert buf.data_ptr() % 256 == 0
        with torch.cuda.device(self.device):
            _check(lib().mcb_build_structure(self._h, which, buf.data_ptr(), nbytes, _stream_ptr(stream)), "mcb_build_structure")
        self._buffers[which] = buf
        return buf

    def drop_structure(self, which: int):
        _torch().cuda.synchronize(self.device)
        _check(lib().mcb_detach_structure(self._h, which), "mcb_detach_structure")
        self._buffers.pop(which, None)

    def fock_export(self, b0: int, count: int, removed: int = 0) -> np.ndarray:
        out = np.empty((count, self.M), dtype=np.int32)
        _check(lib().mcb_fock_export(self._h, removed, b0, count, out.ctypes.data), "mcb_fock_export")
        return out

    def map1_export(self, b0: int, count: int) -> np.ndarray:
        out = np.empty((count, self.M, self.M), dtype=np.int32)
        _check(lib().mcb_map1_export(self._h, b0, count, out.ctypes.data), "mcb_map1_export")
        return out

    def map2_export(self, b0: int, count: int) -> np.ndarray:
        out = np.empty((count, self.P, self.P), dtype=np.int32)
        _check(lib().mcb_map2_export(self._h, b0, count, out.ctypes.data), "mcb_map2_export")
        return out

    def map2c_export(self, b0: int, count: int):
        """(offsets int64 [count + 1], strides int32 [n_strides, P]) of lines b0 .. b0 + count - 1 of the compact double-jump
        map: line b holds the strides offsets[b - b0] - offsets[0] .. offsets[b - b0 + 1] - offsets[0] - 1 of the second array."""
        off = np.empty(count + 1, dtype=np.int64)
        probe = np.empty(1, dtype=np.int32)
        st = lib().mcb_map2c_export(self._h, b0, count, off.ctypes.data, probe.ctypes.data, 0)
        if st not in (OK, ENOMEM):
            raise McbError(st, "mcb_map2c_export")
        n = int(off[count] - off[0])
        ent = np.empty((n, self.P), dtype=np.int32)
        if n > 0:
            _check(lib().mcb_map2c_export(self._h, b0, count, off.ctypes.data, ent.ctypes.data, n * self.P), "mcb_map2c_export")
        return off, ent

    # -- H.C ----------------------------------------------------------------------------------------------
    def apply_workspace_bytes(self, mode: int = AUTO) -> int:
        n = int(lib().mcb_apply_workspace_bytes(self._h, mode))
        if n < 0:
            raise McbError(n, "mcb_apply_workspace_bytes")
        return n

    def _ws(self, mode: int):
        torch = _torch()
        n = self.apply_workspace_bytes(mode)
        if n == 0:
            return 0
        w = self._workspace.get("ws")
        if w is None or w.numel() < n:
            w = torch.empty(n, dtype=torch.uint8, device=self.device)
            self._workspace["ws"] = w
        return w.data_ptr()

    def _check_vec(self, t, name: str):
        """A device vector handed to the library: contiguous complex128, nc elements, on this space's device."""
        torch = _torch()
        if (not isinstance(t, torch.Tensor) or t.dtype != torch.complex128 or not t.is_cuda or not t.is_contiguous()
                or t.numel() != self.nc or t.device != self.device):
            raise ValueError(f"{name} must be a contiguous complex128 CUDA tensor of length nc = {self.nc} on {self.device}")

    def resolve_mode(self, T, V, mode: int = AUTO) -> int:
        """The mode hc_apply will run for these matrix elements (MCB_AUTO looks at their non-zero pattern)."""
        T = _host_c128(T, (self.M, self.M))
        V = _host_c128(V, (self.M,) * 4)
        r = lib().mcb_resolve_mode(self._h, T.ctypes.data, V.ctypes.data, mode)
        if r < 0:
            raise McbError(int(r), "mcb_resolve_mode")
        return int(r)

    def hc_apply(self, T, V, C, out=None, mode: int = AUTO, stream=None):
        """HC = H.C for a complex128 device tensor C [nc]; T [M,M], V [M,M,M,M] host arrays."""
        torch = _torch()
        T = _host_c128(T, (self.M, self.M))
        V = _host_c128(V, (self.M,) * 4)
        self._check_vec(C, "C")
        if out is None:
            out = torch.empty_like(C)
        self._check_vec(out, "out")
        with torch.cuda.device(self.device):
            _check(lib().mcb_hc_apply(self._h, T.ctypes.data, V.ctypes.data, C.data_ptr(), out.data_ptr(), mode,
                                      self._ws(mode), _stream_ptr(stream)), "mcb_hc_apply")
        return out

    def hc_apply_host(self, T, V, C_host, out_host=None, mode: int = AUTO, stream=None):
        """Same through host memory: C_host / out_host are complex128 CPU tensors (pinned for full PCIe speed)
        or numpy arrays.  Copies H2D, applies, copies D2H, synchronises."""
        torch = _torch()
        T = _host_c128(T, (self.M, self.M))
        V = _host_c128(V, (self.M,) * 4)
        if isinstance(C_host, np.ndarray):
            C_host = torch.from_numpy(np.ascontiguousarray(C_host, dtype=np.complex128))
        if C_host.numel() != self.nc or C_host.dtype != torch.complex128 or C_host.is_cuda or not C_host.is_contiguous():
            raise ValueError("C_host must be a contiguous complex128 CPU tensor of length nc")
        if out_host is None:
            out_host = torch.empty_like(C_host)
        if (not isinstance(out_host, torch.Tensor) or out_host.numel() != self.nc or out_host.dtype != torch.complex128
                or out_host.is_cuda or not out_host.is_contiguous()):
            raise ValueError("out_host must be a contiguous complex128 CPU tensor of length nc")
        for name in ("dC", "dHC"):
            if name not in self._workspace:
                self._workspace[name] = torch.empty(self.nc, dtype=torch.complex128, device=self.device)
        with torch.cuda.device(self.device):
            _check(lib().mcb_hc_apply_host(self._h, T.ctypes.data, V.ctypes.data, C_host.data_ptr(), out_host.data_ptr(),
                                           mode, self._workspace["dC"].data_ptr(), self._workspace["dHC"].data_ptr(),
                                           self._ws(mode), _stream_ptr(stream)), "mcb_hc_apply_host")
        return out_host

    def rho(self, C, stream=None):
        """(rho1 [M,M], rho2 [M,M,M,M]) complex128 device tensors: <a+_k a_l>, <a+_k a+_s a_q a_l> of the state C."""
        torch = _torch()
        self._check_vec(C, "C")
        need = lib().mcb_rho_workspace_bytes(self._h)
        if need < 0:
            raise McbError(int(need), "mcb_rho_workspace_bytes")
        ws = self._workspace.get("rho")
        if ws is None or ws.numel() < need:
            ws = self._workspace["rho"] = torch.empty(int(need), dtype=torch.uint8, device=self.device)
        r1 = torch.empty((self.M, self.M), dtype=torch.complex128, device=self.device)
        r2 = torch.empty((self.M,) * 4, dtype=torch.complex128, device=self.device)
        with torch.cuda.device(self.device):
            _check(lib().mcb_rho(self._h, C.data_ptr(), r1.data_ptr(), r2.data_ptr(), ws.data_ptr(), _stream_ptr(stream)), "mcb_rho")
        return r1, r2

    def rho_static(self, C, rho1=None, rho2=None, stream=None):
        """mcb_rho_static: the density matrices of `rho` for callers that cannot allocate device memory -- code that is
        handed its buffers by a host program, runs under a pool that already owns the whole device, or sits in a loop where
        cudaMalloc's device-wide synchronisation is not acceptable.  No workspace is passed: the kernels' scratch is a fixed
        8 MiB array inside libmcb.so (M <= RHO_STATIC_MAX_M = 12; McbError with status ESCRATCH beyond).  Pass `rho1` [M,M] and
        `rho2` [M,M,M,M] (contiguous complex128 CUDA tensors) to keep this Python layer from allocating too; they are created
        here only when left out.  The first call on a device does a one-time address look-up: make it during set-up.  All
        calls on a device share the array -- keep them ordered on one stream (overlapping calls race)."""
        torch = _torch()
        self._check_vec(C, "C")
        outs = []
        for t, shape, name in ((rho1, (self.M, self.M), "rho1"), (rho2, (self.M,) * 4, "rho2")):
            if t is None:
                t = torch.empty(shape, dtype=torch.complex128, device=self.device)
            elif (not isinstance(t, torch.Tensor) or t.dtype != torch.complex128 or not t.is_cuda or not t.is_contiguous()
                    or tuple(t.shape) != shape or t.device != self.device):
                raise ValueError(f"{name} must be a contiguous complex128 CUDA tensor of shape {shape} on {self.device}")
            outs.append(t)
        with torch.cuda.device(self.device):
            _check(lib().mcb_rho_static(self._h, C.data_ptr(), outs[0].data_ptr(), outs[1].data_ptr(), _stream_ptr(stream)),
                   "mcb_rho_static")
        return outs[0], outs[1]

    def lanczos_steps(self, kmax: int = 0) -> int:
        """Steps mcb_lanczos takes for `kmax` (0: the paper's cap nc / 8, at most 1024)."""
        r = int(lib().mcb_lanczos_steps(self._h, kmax))
        if r < 0:
            raise McbError(r, "mcb_lanczos_steps")
        return r

    def lanczos(self, T, V, v0, kmax: int = 0, mode: int = AUTO, breakdown: float = 1e-12, stream=None):
        """(alpha [k], beta [k]) of the Lanczos tridiagonalisation of H started at the device vector v0 (k <= kmax steps;
        kmax = 0: the paper's nc / 8).  tridiag_eigvals(alpha, beta[:-1]) gives the Ritz values.  After the call
        `self.lanczos_truncated` says whether a kmax = 0 run was cut below nc / 8 by the library's cap (MCB_TRUNCATED)."""
        torch = _torch()
        T = _host_c128(T, (self.M, self.M))
        V = _host_c128(V, (self.M,) * 4)
        self._check_vec(v0, "v0")
        need = lib().mcb_lanczos_workspace_bytes(self._h, kmax)
        if need < 0:
            raise McbError(int(need), "mcb_lanczos_workspace_bytes")
        ws = self._workspace.get("lanczos")
        if ws is None or ws.numel() < need:
            ws = self._workspace["lanczos"] = torch.empty(int(need), dtype=torch.uint8, device=self.device)
        steps = self.lanczos_steps(kmax)
        alpha = np.zeros(steps, dtype=np.float64)
        beta = np.zeros(steps, dtype=np.float64)
        k = ctypes.c_int(0)
        with torch.cuda.device(self.device):
            status = lib().mcb_lanczos(self._h, T.ctypes.data, V.ctypes.data, v0.data_ptr(), kmax, mode, breakdown,
                                       alpha.ctypes.data, beta.ctypes.data, ctypes.byref(k), ws.data_ptr(), self._ws(mode),
                                       _stream_ptr(stream))
        self.lanczos_truncated = status == TRUNCATED
        if status != TRUNCATED:
            _check(status, "mcb_lanczos")
        return alpha[:k.value], beta[:k.value]

    def timing_enable(self, on: bool = True):
        _check(lib().mcb_timing_enable(self._h, 1 if on else 0), "mcb_timing_enable")

    def timing_read(self, max_applies: int = 512):
        """(ms [applies, 3] float32, launches [applies] int32) of the applies recorded since timing_enable."""
        ms = np.zeros((max_applies, 3), dtype=np.float32)
        la = np.zeros(max_applies, dtype=np.int32)
        n = lib().mcb_timing_read(self._h, max_applies, ms.ctypes.data, la.ctypes.data)
        if n < 0:
            raise McbError(n, "mcb_timing_read")
        return ms[:n], la[:n]

    def debug_bounds(self):
        """(compiled_in, site, index): the library's own bounds checks (builds with -DMCB_DEBUG_BOUNDS); site 0 = no violation."""
        out = np.zeros(2, dtype=np.int64)
        r = lib().mcb_debug_bounds(self._h, out.ctypes.data)
        if r < 0:
            raise McbError(int(r), "mcb_debug_bounds")
        return bool(r), int(out[0]), int(out[1])

    def last_apply_launches(self) -> int:
        return int(lib().mcb_last_apply_launches(self._h))

    def last_apply_memops(self):
        """(memcpy, memset) operations the last hc_apply enqueued beside its kernels, as counted by the library."""
        a, b = ctypes.c_int(0), ctypes.c_int(0)
        _check(lib().mcb_last_apply_memops(self._h, ctypes.byref(a), ctypes.byref(b)), "mcb_last_apply_memops")
        return int(a.value), int(b.value)
