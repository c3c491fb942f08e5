"""Thin ctypes binding of the C-ABI library (include/berryeasy_b200.h).

Argument marshalling only: every step of the path runs in the CUDA kernels of
``libberryeasy_b200.so``.  PyTorch supplies device memory and streams.  There is no CPU fallback:
if the library is missing or no CUDA device is present the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libberryeasy_b200.so")

EXPORTS = [
    "be_create", "be_destroy", "be_strerror", "be_workspace_bytes", "be_set_workspace_limit",
    "be_launch_count", "be_host_grid_bytes_copied", "be_host_schedule", "be_eigh_batched", "be_eigh_batched_static", "be_wilson_loop", "be_nested_wilson",
    "be_spin_resolved_wilson", "be_winding", "be_wilson_loop_host", "be_spin_resolved_wilson_host", "be_nested_wilson_host",
    "be_profile_enable", "be_profile_name", "be_profile_get", "be_zgemm_batched", "be_set_chunk_pipeline", "be_set_eigh_algorithm", "be_probe_fp64", "be_release_workspace", "be_bloch_coefficients", "be_assemble_bloch", "be_plaquette_flux", "be_wilson_loop_bloch",
    "be_spin_resolved_wilson_bloch", "be_wilson_loop_window", "be_spin_resolved_wilson_window",
]


class BeGrid(C.Structure):
    _fields_ = [("ndim", C.c_int), ("batch", C.c_int64), ("dims", C.c_int * 3), ("N", C.c_int)]


_lib = None


def load_library():
    """dlopen the in-tree shared library (built by ``python -m paper_2312_13051_b200.build``)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} not found: run `python -m paper_2312_13051_b200.build` "
                           "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, i64, dbl, ci = C.c_void_p, C.c_int64, C.c_double, C.c_int
    gp = C.POINTER(BeGrid)
    lib.be_create.argtypes = [C.POINTER(vp), vp]
    lib.be_destroy.argtypes = [vp]
    lib.be_strerror.argtypes = [ci]
    lib.be_strerror.restype = C.c_char_p
    lib.be_workspace_bytes.argtypes = [gp, ci, ci]
    lib.be_workspace_bytes.restype = C.c_size_t
    lib.be_set_workspace_limit.argtypes = [vp, C.c_size_t]
    lib.be_set_chunk_pipeline.argtypes = [vp, ci]
    lib.be_set_eigh_algorithm.argtypes = [vp, ci]
    lib.be_probe_fp64.argtypes = [vp, ci, C.POINTER(dbl)]
    lib.be_release_workspace.argtypes = [vp]
    lib.be_bloch_coefficients.argtypes = [vp, vp, C.POINTER(ci), ci, ci, i64, vp]
    lib.be_assemble_bloch.argtypes = [vp, vp, vp, i64, ci, ci, vp]
    lib.be_plaquette_flux.argtypes = [vp, vp, gp, ci, vp, ci, ci, vp, vp, vp]
    lib.be_wilson_loop_bloch.argtypes = [vp, vp, C.POINTER(ci), ci, gp, ci, ci, vp, vp, vp, vp]
    lib.be_spin_resolved_wilson_bloch.argtypes = [vp, vp, C.POINTER(ci), ci, gp, ci, ci, vp, ci, ci, vp, vp, vp, vp]
    lib.be_launch_count.argtypes = [vp]
    lib.be_launch_count.restype = i64
    lib.be_host_grid_bytes_copied.argtypes = [vp]
    lib.be_host_grid_bytes_copied.restype = i64
    lib.be_host_schedule.argtypes = [vp]
    lib.be_host_schedule.restype = ci
    lib.be_eigh_batched.argtypes = [vp, vp, i64, ci, ci, vp, vp, vp]
    lib.be_eigh_batched_static.argtypes = [vp, vp, i64, ci, ci, vp, vp, vp]
    lib.be_wilson_loop.argtypes = [vp, vp, gp, ci, ci, vp, vp, vp, vp]
    lib.be_wilson_loop_window.argtypes = [vp, vp, gp, ci, ci, ci, vp, vp, vp, vp]
    lib.be_spin_resolved_wilson_window.argtypes = [vp, vp, gp, ci, ci, ci, vp, ci, ci, vp, vp, vp, vp]
    lib.be_nested_wilson.argtypes = [vp, vp, gp, ci, ci, ci, ci, ci, ci, dbl, vp, vp, vp, vp]
    lib.be_spin_resolved_wilson.argtypes = [vp, vp, gp, ci, ci, vp, ci, ci, vp, vp, vp, vp]
    lib.be_winding.argtypes = [vp, vp, i64, ci, ci, vp]
    lib.be_wilson_loop_host.argtypes = [vp, vp, gp, ci, ci, vp, vp, vp, vp]
    lib.be_spin_resolved_wilson_host.argtypes = [vp, vp, gp, ci, ci, vp, ci, ci, vp, vp, vp, vp]
    lib.be_nested_wilson_host.argtypes = [vp, vp, gp, ci, ci, ci, ci, ci, ci, dbl, vp, vp, vp, vp]
    lib.be_zgemm_batched.argtypes = [vp, ci, ci, ci, ci, ci, C.POINTER(dbl), vp, ci, i64, vp, ci, i64,
                                     C.POINTER(dbl), vp, ci, i64, i64, ci]
    lib.be_profile_enable.argtypes = [vp, ci]
    lib.be_profile_name.argtypes = [ci]
    lib.be_profile_name.restype = C.c_char_p
    lib.be_profile_get.argtypes = [vp, ci, C.POINTER(dbl), C.POINTER(i64), C.POINTER(dbl), C.POINTER(dbl)]
    _lib = lib
    return lib


class BerryEasyError(RuntimeError):
    pass


def _check(lib, rc):
    if rc != 0:
        raise BerryEasyError(f"berryeasy_b200 error {rc}: {lib.be_strerror(rc).decode()}")


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _dev(t, dtype, name):
    if not t.is_cuda:
        raise ValueError(f"{name} must be a CUDA tensor")
    if t.dtype != dtype or not t.is_contiguous():
        raise ValueError(f"{name} must be contiguous {dtype}")
    return t


def _host(t, dtype, name):
    if t.is_cuda or t.dtype != dtype or not t.is_contiguous():
        raise ValueError(f"{name} must be a contiguous host tensor of {dtype}")
    return t


def _grid_of(H, grid_ndim):
    if H.dim() != grid_ndim + 3:
        raise ValueError("H_grid must be [batch][dims...][N][N]")
    g = BeGrid()
    g.ndim = grid_ndim
    g.batch = H.shape[0]
    for a in range(3):
        g.dims[a] = H.shape[1 + a] if a < grid_ndim else 1
    g.N = H.shape[-1]
    if H.shape[-2] != H.shape[-1]:
        raise ValueError("H must be square")
    return g


class Context:
    """Owns a ``be_ctx`` bound to the current torch CUDA stream (or the one given)."""

    def __init__(self, stream: "torch.cuda.Stream | None" = None, device=None):
        if not torch.cuda.is_available():
            raise RuntimeError("berryeasy_b200 needs a CUDA device (no CPU fallback)")
        self.lib = load_library()
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        with torch.cuda.device(self.device):
            self.stream = stream if stream is not None else torch.cuda.current_stream()
            h = C.c_void_p()
            _check(self.lib, self.lib.be_create(C.byref(h), C.c_void_p(self.stream.cuda_stream)))
        self._h = h

    def close(self):
        if getattr(self, "_h", None):
            self.lib.be_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_workspace_limit(self, nbytes: int):
        _check(self.lib, self.lib.be_set_workspace_limit(self._h, nbytes))

    def set_chunk_pipeline(self, on: bool):
        _check(self.lib, self.lib.be_set_chunk_pipeline(self._h, 1 if on else 0))

    def set_eigh_algorithm(self, algo: int):
        """0: one-stage tridiagonalization, 1: two-stage (dense -> band -> tridiagonal) where supported."""
        _check(self.lib, self.lib.be_set_eigh_algorithm(self._h, int(algo)))

    def release_workspace(self):
        """Give the scratch arena and the staging buffers back to the device (re-allocated on demand)."""
        _check(self.lib, self.lib.be_release_workspace(self._h))

    def probe_fp64(self) -> dict:
        """Measured FP64 rates of this device under the current clocks (TFLOP/s): DMMA chain, DFMA chain with
        operand reuse, DFMA chain with three distinct register operands."""
        out = {}
        for which, name in ((0, "dmma"), (1, "dfma"), (2, "dfma_3operand")):
            v = C.c_double()
            _check(self.lib, self.lib.be_probe_fp64(self._h, which, C.byref(v)))
            out[name] = v.value
        return out

    def profile_enable(self, on: bool = True):
        _check(self.lib, self.lib.be_profile_enable(self._h, 1 if on else 0))

    def profile(self) -> dict:
        """{class: {ms, launches, bytes, flops}} summed since profile_enable."""
        out = {}
        i = 0
        while True:
            name = self.lib.be_profile_name(i)
            if not name:
                break
            ms, n, by, fl = C.c_double(), C.c_int64(), C.c_double(), C.c_double()
            _check(self.lib, self.lib.be_profile_get(self._h, i, C.byref(ms), C.byref(n), C.byref(by), C.byref(fl)))
            out[name.decode()] = {"ms": ms.value, "launches": n.value, "bytes": by.value, "flops": fl.value}
            i += 1
        return out

    def launch_count(self) -> int:
        return int(self.lib.be_launch_count(self._h))

    def host_schedule(self) -> int:
        """n > 0: the last *_host call ran n chunks; n < 0: one chunk fed in -n sub-ranges (be_host_schedule)."""
        return int(self.lib.be_host_schedule(self._h))

    def host_grid_bytes_copied(self) -> int:
        """Bytes of H_grid the *_host calls of this context have copied to the device so far."""
        return int(self.lib.be_host_grid_bytes_copied(self._h))

    # ------------------------------------------------------------------ be_eigh_batched
    def eigh_batched(self, H, n_vec=None, want_info=False):
        """H [count][N][N] complex128 (device) -> E [count][N], U [count][N][n_vec] (or None)."""
        _dev(H, torch.complex128, "H")
        count, N = H.shape[0], H.shape[-1]
        n_vec = N if n_vec is None else n_vec
        E = torch.empty((count, N), dtype=torch.float64, device=H.device)
        U = torch.empty((count, N, n_vec), dtype=torch.complex128, device=H.device) if n_vec > 0 else None
        info = torch.empty((count,), dtype=torch.int32, device=H.device) if want_info else None
        _check(self.lib, self.lib.be_eigh_batched(self._h, _ptr(H), count, N, n_vec, _ptr(E), _ptr(U), _ptr(info)))
        return (E, U, info) if want_info else (E, U)

    def eigh_batched_static(self, H, E, U=None, info=None):
        """be_eigh_batched_static: N <= 8, caller-provided outputs E [count][N], U [count][N][n_vec] or None; the
        library allocates nothing (fixed device scratch, BE_STATIC_EIGH_MAX_ELEMS)."""
        _dev(H, torch.complex128, "H")
        _dev(E, torch.float64, "E")
        count, N = H.shape[0], H.shape[-1]
        n_vec = 0
        if U is not None:
            _dev(U, torch.complex128, "U")
            n_vec = U.shape[-1]
        _check(self.lib, self.lib.be_eigh_batched_static(self._h, _ptr(H), count, N, n_vec, _ptr(E), _ptr(U), _ptr(info)))
        return E, U

    # ------------------------------------------------------------------ be_wilson_loop
    def wilson_loop(self, H_grid, n_occ, direction, close=None, want_abs=True, want_mingap=True, band_lo=0):
        """H_grid [batch][dims...][N][N] -> theta [loops][m], |lambda| or None, mingap or None.

        Bands [band_lo, n_occ) in ascending-energy order (be_wilson_loop_window when band_lo > 0)."""
        if band_lo:
            return self._wilson_loop_window(H_grid, band_lo, n_occ, direction, close, want_abs, want_mingap)
        _dev(H_grid, torch.complex128, "H_grid")
        nd = H_grid.dim() - 3
        g = _grid_of(H_grid, nd)
        loops = H_grid.shape[0]
        for a in range(nd):
            if a != direction:
                loops *= H_grid.shape[1 + a]
        dev = H_grid.device
        theta = torch.empty((loops, n_occ), dtype=torch.float64, device=dev)
        ab = torch.empty((loops, n_occ), dtype=torch.float64, device=dev) if want_abs else None
        mg = torch.empty((loops,), dtype=torch.float64, device=dev) if want_mingap else None
        if close is not None:
            _dev(close, torch.complex128, "close")
        _check(self.lib, self.lib.be_wilson_loop(self._h, _ptr(H_grid), C.byref(g), n_occ, direction,
                                                 _ptr(close), _ptr(theta), _ptr(ab), _ptr(mg)))
        return theta, ab, mg

    def _wilson_loop_window(self, H_grid, band_lo, band_hi, direction, close, want_abs, want_mingap):
        _dev(H_grid, torch.complex128, "H_grid")
        nd = H_grid.dim() - 3
        g = _grid_of(H_grid, nd)
        loops = H_grid.shape[0]
        for a in range(nd):
            if a != direction:
                loops *= H_grid.shape[1 + a]
        dev = H_grid.device
        m = max(band_hi - band_lo, 0)
        theta = torch.empty((loops, m), dtype=torch.float64, device=dev)
        ab = torch.empty((loops, m), dtype=torch.float64, device=dev) if want_abs else None
        mg = torch.empty((loops,), dtype=torch.float64, device=dev) if want_mingap else None
        if close is not None:
            _dev(close, torch.complex128, "close")
        _check(self.lib, self.lib.be_wilson_loop_window(self._h, _ptr(H_grid), C.byref(g), band_lo, band_hi, direction,
                                                        _ptr(close), _ptr(theta), _ptr(ab), _ptr(mg)))
        return theta, ab, mg

    def spin_resolved_wilson_window(self, H_grid, band_lo, band_hi, direction, S, m_lo=-1, close=None, want_pso=True):
        """be_spin_resolved_wilson_window: the spin-resolved loop of the bands [band_lo, band_hi)."""
        _dev(H_grid, torch.complex128, "H_grid")
        nd = H_grid.dim() - 3
        g = _grid_of(H_grid, nd)
        loops = H_grid.shape[0]
        for a in range(nd):
            if a != direction:
                loops *= H_grid.shape[1 + a]
        n1 = H_grid.shape[1 + direction]
        is_diag = 1 if S.dim() == 1 else 0
        _dev(S, torch.float64 if is_diag else torch.complex128, "S")
        m = max(band_hi - band_lo, 0)
        mlo = m // 2 if m_lo < 0 else m_lo
        dev = H_grid.device
        lo = torch.empty((loops, mlo), dtype=torch.float64, device=dev)
        hi = torch.empty((loops, max(m - mlo, 0)), dtype=torch.float64, device=dev)
        pso = torch.empty((loops, n1, m), dtype=torch.float64, device=dev) if want_pso else None
        _check(self.lib, self.lib.be_spin_resolved_wilson_window(self._h, _ptr(H_grid), C.byref(g), band_lo, band_hi,
                                                                 direction, _ptr(S), is_diag, m_lo, _ptr(close),
                                                                 _ptr(lo), _ptr(hi), _ptr(pso)))
        return lo, hi, pso

    # ------------------------------------------------------------------ be_spin_resolved_wilson
    def spin_resolved_wilson(self, H_grid, n_occ, direction, S, m_lo=-1, close=None, want_pso=True):
        """S: real diagonal [N] float64 or dense [N][N] complex128 (device)."""
        _dev(H_grid, torch.complex128, "H_grid")
        nd = H_grid.dim() - 3
        g = _grid_of(H_grid, nd)
        loops = H_grid.shape[0]
        for a in range(nd):
            if a != direction:
                loops *= H_grid.shape[1 + a]
        n1 = H_grid.shape[1 + direction]
        is_diag = 1 if S.dim() == 1 else 0
        _dev(S, torch.float64 if is_diag else torch.complex128, "S")
        mlo = n_occ // 2 if m_lo < 0 else m_lo
        dev = H_grid.device
        lo = torch.empty((loops, mlo), dtype=torch.float64, device=dev)
        hi = torch.empty((loops, n_occ - mlo), dtype=torch.float64, device=dev)
        pso = torch.empty((loops, n1, n_occ), dtype=torch.float64, device=dev) if want_pso else None
        _check(self.lib, self.lib.be_spin_resolved_wilson(self._h, _ptr(H_grid), C.byref(g), n_occ, direction,
                                                          _ptr(S), is_diag, m_lo, _ptr(close),
                                                          _ptr(lo), _ptr(hi), _ptr(pso)))
        return lo, hi, pso

    # ------------------------------------------------------------------ be_nested_wilson
    def nested_wilson(self, H_grid, n_occ, dir1, dir2, base=0, wb_lo=0, wb_hi=1, theta_cut=None,
                      close1=None, close2=None):
        import math
        _dev(H_grid, torch.complex128, "H_grid")
        nd = H_grid.dim() - 3
        g = _grid_of(H_grid, nd)
        outer = H_grid.shape[0]
        for a in range(nd):
            if a not in (dir1, dir2):
                outer *= H_grid.shape[1 + a]
        n2 = H_grid.shape[1 + dir2]
        dev = H_grid.device
        th1 = torch.empty((outer, n2, n_occ), dtype=torch.float64, device=dev)
        thn = torch.empty((outer, wb_hi - wb_lo), dtype=torch.float64, device=dev)
        cut = math.pi if theta_cut is None else float(theta_cut)
        _check(self.lib, self.lib.be_nested_wilson(self._h, _ptr(H_grid), C.byref(g), n_occ, dir1, dir2, base,
                                                   wb_lo, wb_hi, cut, _ptr(close1), _ptr(close2),
                                                   _ptr(th1), _ptr(thn)))
        return th1, thn

    # ------------------------------------------------------------------ be_zgemm_batched
    def zgemm_batched(self, opA, opB, A, B, C_out, M, N, K, lda, ldb, ldc, strideA, strideB, strideC, batch,
                      alpha=1.0 + 0j, beta=0.0 + 0j, lower=False):
        """Raw column-major batched GEMM on device tensors (complex128).  ops: 'N','T','C','J'."""
        ops = {"N": 0, "T": 1, "C": 2, "J": 3}
        al = (C.c_double * 2)(alpha.real, alpha.imag)
        be = (C.c_double * 2)(beta.real, beta.imag)
        _check(self.lib, self.lib.be_zgemm_batched(self._h, ops[opA], ops[opB], M, N, K, al, _ptr(A), lda, strideA,
                                                   _ptr(B), ldb, strideB, be, _ptr(C_out), ldc, strideC, batch,
                                                   1 if lower else 0))
        return C_out

    # ------------------------------------------------------------------ H(k) assembly (NEXT-1)
    def assemble_bloch(self, A, t, R):
        """A [nR][N][N] complex128 blocks (device), t [count][nd] float64 reduced coordinates (device),
        R [nR][nd] ints (host list / array) -> H [count][N][N] = sum_R exp(2 pi i t.R) A_R."""
        _dev(A, torch.complex128, "A")
        _dev(t, torch.float64, "t")
        nR, N = A.shape[0], A.shape[-1]
        count, nd = t.shape
        Rl = [int(x) for row in R for x in row]
        if len(Rl) != nR * nd:
            raise ValueError("R must be [nR][nd]")
        hR = (C.c_int * len(Rl))(*Rl)
        coef = torch.empty((count, nR), dtype=torch.complex128, device=A.device)
        _check(self.lib, self.lib.be_bloch_coefficients(self._h, _ptr(t), hR, nd, nR, count, _ptr(coef)))
        H = torch.empty((count, N, N), dtype=torch.complex128, device=A.device)
        _check(self.lib, self.lib.be_assemble_bloch(self._h, _ptr(A), _ptr(coef), count, N, nR, _ptr(H)))
        return H

    # ------------------------------------------------------------------ fused H(k) generation (NEXT-1)
    def _bloch_grid(self, A, dims):
        if A.dim() != 4:
            raise ValueError("A must be [batch][nR][N][N]")
        g = BeGrid()
        g.ndim = len(dims)
        g.batch = A.shape[0]
        for a in range(3):
            g.dims[a] = dims[a] if a < len(dims) else 1
        g.N = A.shape[-1]
        return g

    def wilson_loop_bloch(self, A, R, dims, n_occ, direction, close=None):
        """A [batch][nR][N][N] blocks (device), R [nR][ndim] ints, dims = grid points per axis: the loops of
        be_wilson_loop on the grid H = sum_R exp(2 pi i (i/dims).R) A_R, generated on the fly."""
        _dev(A, torch.complex128, "A")
        g = self._bloch_grid(A, dims)
        nR = A.shape[1]
        Rl = [int(x) for row in R for x in row]
        if len(Rl) != nR * len(dims):
            raise ValueError("R must be [nR][ndim]")
        hR = (C.c_int * len(Rl))(*Rl)
        loops = A.shape[0]
        for a, d in enumerate(dims):
            if a != direction:
                loops *= d
        dev = A.device
        theta = torch.empty((loops, n_occ), dtype=torch.float64, device=dev)
        ab = torch.empty((loops, n_occ), dtype=torch.float64, device=dev)
        mg = torch.empty((loops,), dtype=torch.float64, device=dev)
        _check(self.lib, self.lib.be_wilson_loop_bloch(self._h, _ptr(A), hR, nR, C.byref(g), n_occ, direction,
                                                       _ptr(close), _ptr(theta), _ptr(ab), _ptr(mg)))
        return theta, ab, mg

    def spin_resolved_wilson_bloch(self, A, R, dims, n_occ, direction, S, m_lo=-1, close=None):
        _dev(A, torch.complex128, "A")
        g = self._bloch_grid(A, dims)
        nR = A.shape[1]
        Rl = [int(x) for row in R for x in row]
        hR = (C.c_int * len(Rl))(*Rl)
        loops = A.shape[0]
        for a, d in enumerate(dims):
            if a != direction:
                loops *= d
        n1 = dims[direction]
        is_diag = 1 if S.dim() == 1 else 0
        _dev(S, torch.float64 if is_diag else torch.complex128, "S")
        mlo = n_occ // 2 if m_lo < 0 else m_lo
        dev = A.device
        lo = torch.empty((loops, mlo), dtype=torch.float64, device=dev)
        hi = torch.empty((loops, n_occ - mlo), dtype=torch.float64, device=dev)
        pso = torch.empty((loops, n1, n_occ), dtype=torch.float64, device=dev)
        _check(self.lib, self.lib.be_spin_resolved_wilson_bloch(self._h, _ptr(A), hR, nR, C.byref(g), n_occ, direction,
                                                                _ptr(S), is_diag, m_lo, _ptr(close), _ptr(lo),
                                                                _ptr(hi), _ptr(pso)))
        return lo, hi, pso

    # ------------------------------------------------------------------ be_plaquette_flux (NEXT-2)
    def plaquette_flux(self, H_grid, n_occ, S=None, m_lo=-1, want_pso=False):
        """H_grid [batch][ny][nx][N][N] (device) -> flux [batch][ny][nx]; with S: (flux_lo, flux_hi[, pso])."""
        _dev(H_grid, torch.complex128, "H_grid")
        if H_grid.dim() != 5:
            raise ValueError("H_grid must be [batch][ny][nx][N][N]")
        g = _grid_of(H_grid, 2)
        shp = tuple(H_grid.shape[:3])
        dev = H_grid.device
        f0 = torch.empty(shp, dtype=torch.float64, device=dev)
        if S is None:
            _check(self.lib, self.lib.be_plaquette_flux(self._h, _ptr(H_grid), C.byref(g), n_occ, None, 0, -1,
                                                        _ptr(f0), None, None))
            return f0
        is_diag = 1 if S.dim() == 1 else 0
        _dev(S, torch.float64 if is_diag else torch.complex128, "S")
        f1 = torch.empty(shp, dtype=torch.float64, device=dev)
        pso = torch.empty(shp + (n_occ,), dtype=torch.float64, device=dev) if want_pso else None
        _check(self.lib, self.lib.be_plaquette_flux(self._h, _ptr(H_grid), C.byref(g), n_occ, _ptr(S), is_diag, m_lo,
                                                    _ptr(f0), _ptr(f1), _ptr(pso)))
        return (f0, f1, pso) if want_pso else (f0, f1)

    # ------------------------------------------------------------------ be_winding
    def winding(self, theta):
        """theta [n_cycles][n_points][m] (device) -> wind [n_cycles]."""
        _dev(theta, torch.float64, "theta")
        nc, npnt, m = theta.shape
        out = torch.empty((nc,), dtype=torch.float64, device=theta.device)
        _check(self.lib, self.lib.be_winding(self._h, _ptr(theta), nc, npnt, m, _ptr(out)))
        return out

    # ------------------------------------------------------------------ host variants (end to end)
    def wilson_loop_host(self, H_grid, n_occ, direction, close=None):
        _host(H_grid, torch.complex128, "H_grid")
        nd = H_grid.dim() - 3
        g = _grid_of(H_grid, nd)
        loops = H_grid.numel() // (H_grid.shape[-1] ** 2 * H_grid.shape[1 + direction])
        theta = torch.empty((loops, n_occ), dtype=torch.float64).pin_memory()
        ab = torch.empty((loops, n_occ), dtype=torch.float64).pin_memory()
        mg = torch.empty((loops,), dtype=torch.float64).pin_memory()
        _check(self.lib, self.lib.be_wilson_loop_host(self._h, _ptr(H_grid), C.byref(g), n_occ, direction,
                                                      _ptr(close), _ptr(theta), _ptr(ab), _ptr(mg)))
        return theta, ab, mg

    def spin_resolved_wilson_host(self, H_grid, n_occ, direction, S, m_lo=-1, close=None, want_pso=True):
        _host(H_grid, torch.complex128, "H_grid")
        nd = H_grid.dim() - 3
        g = _grid_of(H_grid, nd)
        n1 = H_grid.shape[1 + direction]
        loops = H_grid.numel() // (H_grid.shape[-1] ** 2 * n1)
        is_diag = 1 if S.dim() == 1 else 0
        mlo = n_occ // 2 if m_lo < 0 else m_lo
        lo = torch.empty((loops, mlo), dtype=torch.float64).pin_memory()
        hi = torch.empty((loops, n_occ - mlo), dtype=torch.float64).pin_memory()
        pso = torch.empty((loops, n1, n_occ), dtype=torch.float64).pin_memory() if want_pso else None
        _check(self.lib, self.lib.be_spin_resolved_wilson_host(self._h, _ptr(H_grid), C.byref(g), n_occ,
                                                               direction, _ptr(S), is_diag, m_lo, _ptr(close),
                                                               _ptr(lo), _ptr(hi), _ptr(pso)))
        return lo, hi, pso

    def nested_wilson_host(self, H_grid, n_occ, dir1, dir2, base=0, wb_lo=0, wb_hi=1, theta_cut=None,
                           close1=None, close2=None):
        import math
        _host(H_grid, torch.complex128, "H_grid")
        nd = H_grid.dim() - 3
        g = _grid_of(H_grid, nd)
        outer = H_grid.shape[0]
        for a in range(nd):
            if a not in (dir1, dir2):
                outer *= H_grid.shape[1 + a]
        n2 = H_grid.shape[1 + dir2]
        th1 = torch.empty((outer, n2, n_occ), dtype=torch.float64).pin_memory()
        thn = torch.empty((outer, wb_hi - wb_lo), dtype=torch.float64).pin_memory()
        cut = math.pi if theta_cut is None else float(theta_cut)
        _check(self.lib, self.lib.be_nested_wilson_host(self._h, _ptr(H_grid), C.byref(g), n_occ, dir1, dir2, base,
                                                        wb_lo, wb_hi, cut, _ptr(close1), _ptr(close2),
                                                        _ptr(th1), _ptr(thn)))
        return th1, thn
