"""Thin ctypes binding of the C-ABI library (include/wilson_cg.h) — argument marshalling only.

Every step of the path runs in the CUDA kernels behind the ABI; there is no CPU fallback: if the
shared object is missing this module raises at first use (build it with
`python -m paper_2111_14958_b200.build`).  PyTorch is used for device memory and streams only.

Names follow the header: wd_create -> WilsonContext, wd_apply -> .wd_apply, cg_solve -> .cg_solve, ...
"""
from __future__ import annotations

import ctypes
import os
import re

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libwilson_cg.so")
HEADER_PATH = os.path.join(os.path.dirname(HERE), "include", "wilson_cg.h")

WD_OK = 0
WD_NOT_CONVERGED = 1
WD_BREAKDOWN = 2

_lib = None


class WdCgInfo(ctypes.Structure):
    _fields_ = [
        ("iterations", ctypes.c_int),
        ("converged", ctypes.c_int),
        ("rel_residual", ctypes.c_double),
        ("eta_norm2", ctypes.c_double),
        ("gpu_ms", ctypes.c_double),
        ("total_ms", ctypes.c_double),
        ("kernel_launches", ctypes.c_int),
        ("cg_mode", ctypes.c_int),
    ]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_ if k != "_"}


class WilsonError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"wilson_cg error {code}: {msg}")
        self.code = code


def declared_symbols(header_path: str = HEADER_PATH):
    """Function names declared in include/wilson_cg.h (used by the symbol-export test)."""
    text = open(header_path).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b((?:wd|cg|bicgstab)_[a-z0-9_]+)\s*\(", text)))


def load_library(path: str = LIB_PATH):
    """dlopen the library and declare the prototypes.  Raises if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(path):
        raise FileNotFoundError(
            f"{path} not found: build it with `python -m paper_2111_14958_b200.build` (no CPU fallback exists)")
    lib = ctypes.CDLL(path)
    vp, ip, dp = ctypes.c_void_p, ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ctypes.c_double)
    cd, ci = ctypes.c_double, ctypes.c_int
    lib.wd_create.argtypes = [ctypes.POINTER(vp), ip, ci, ci, vp]
    lib.wd_destroy.argtypes = [vp]
    lib.wd_last_error.argtypes = [vp]
    lib.wd_last_error.restype = ctypes.c_char_p
    lib.wd_gauge_native_bytes.argtypes = [vp]
    lib.wd_gauge_native_bytes.restype = ctypes.c_size_t
    lib.wd_spinor_native_bytes.argtypes = [vp]
    lib.wd_spinor_native_bytes.restype = ctypes.c_size_t
    lib.wd_pack_gauge.argtypes = [vp, vp, vp]
    lib.wd_pack_spinor.argtypes = [vp, vp, vp]
    lib.wd_unpack_spinor.argtypes = [vp, vp, vp]
    lib.wd_apply.argtypes = [vp, vp, vp, vp, cd, ci]
    lib.cg_solve.argtypes = [vp, vp, vp, vp, cd, cd, ci, ctypes.POINTER(WdCgInfo)]
    lib.bicgstab_solve.argtypes = [vp, vp, vp, vp, cd, cd, ci, ctypes.POINTER(WdCgInfo)]
    lib.wd_get_profile_bicgstab.argtypes = [vp, dp, ctypes.POINTER(ctypes.c_long)]
    lib.wd_eo_spinor_bytes.argtypes = [vp]
    lib.wd_eo_spinor_bytes.restype = ctypes.c_size_t
    lib.wd_eo_gauge_bytes.argtypes = [vp]
    lib.wd_eo_gauge_bytes.restype = ctypes.c_size_t
    lib.wd_eo_pack_spinor.argtypes = [vp, vp, vp]
    lib.wd_eo_unpack_spinor.argtypes = [vp, vp, vp]
    lib.wd_eo_pack_gauge.argtypes = [vp, vp, vp]
    lib.wd_eo_hop.argtypes = [vp, vp, vp, vp, ci, ci]
    lib.cg_solve_eo.argtypes = [vp, vp, vp, vp, cd, cd, ci, ctypes.POINTER(WdCgInfo)]
    lib.bicgstab_solve_eo.argtypes = [vp, vp, vp, vp, cd, cd, ci, ctypes.POINTER(WdCgInfo)]
    lib.wd_get_profile_eo_bicgstab.argtypes = [vp, dp, ctypes.POINTER(ctypes.c_long)]
    lib.wd_apply_multi.argtypes = [vp, vp, vp, vp, ci, cd, ci]
    lib.cg_solve_multi.argtypes = [vp, vp, vp, vp, ci, cd, cd, ci, ctypes.POINTER(WdCgInfo)]
    lib.wd_coo_nnz.argtypes = [vp]
    lib.wd_coo_nnz.restype = ctypes.c_size_t
    lib.wd_coo_assemble.argtypes = [vp, vp, cd, ci, vp, vp, vp]
    lib.wd_coo_spmv.argtypes = [vp, ctypes.c_size_t, vp, vp, vp, vp, vp]
    lib.wd_apply_host.argtypes = [vp, vp, vp, vp, cd, ci]
    lib.wd_apply_repeat.argtypes = [vp, vp, vp, vp, cd, ci, ci, dp]
    lib.cg_solve_host.argtypes = [vp, vp, vp, vp, cd, cd, ci, ctypes.POINTER(WdCgInfo)]
    lib.cg_solve_host_begin.argtypes = [vp, vp, vp]
    lib.cg_solve_host_run.argtypes = [vp, vp, cd, cd, ci, ctypes.POINTER(WdCgInfo)]
    lib.cg_solve_host_wait.argtypes = [vp]
    lib.wd_cg_history.argtypes = [vp, dp, ci]
    lib.wd_norm2.argtypes = [vp, vp, dp]
    lib.wd_norm2_noalloc.argtypes = [ci, ctypes.c_size_t, vp, vp, vp]
    lib.wd_noalloc_max_sites.argtypes = [ci]
    lib.wd_noalloc_max_sites.restype = ctypes.c_size_t
    lib.wd_noalloc_prepare.argtypes = []
    lib.wd_noalloc_last_error.argtypes = []
    lib.wd_noalloc_last_error.restype = ctypes.c_char_p
    lib.wd_num_tiles.argtypes = []
    lib.wd_tile_shape.argtypes = [ci, ip]
    lib.wd_tile_info.argtypes = [ci, ip]
    lib.wd_set_tile.argtypes = [vp, ci]
    lib.wd_get_tile.argtypes = [vp]
    lib.wd_set_cg_mode.argtypes = [vp, ci]
    lib.wd_set_gauge_recon.argtypes = [vp, ci]
    lib.wd_get_gauge_recon.argtypes = [vp]
    lib.wd_set_zchunk.argtypes = [vp, ci]
    lib.wd_set_small_tile.argtypes = [vp, ci]
    lib.wd_set_poll_interval.argtypes = [vp, ci]
    lib.wd_set_coo_fast.argtypes = [vp, ci]
    lib.wd_num_staging_rows.argtypes = []
    lib.wd_staging_row_info.argtypes = [ci, ip]
    lib.wd_set_link_staging.argtypes = [vp, ci]
    lib.wd_get_link_staging.argtypes = [vp]
    lib.wd_set_profile.argtypes = [vp, ci]
    lib.wd_get_profile.argtypes = [vp, dp, ctypes.POINTER(ctypes.c_long)]
    lib.wd_selftest_fastdiv.argtypes = [ctypes.c_uint, ctypes.c_uint]
    lib.wd_selftest_fastdiv.restype = ctypes.c_long
    lib.wd_version.argtypes = []
    lib.wd_version.restype = ctypes.c_char_p
    _lib = lib
    return lib


def tile_shapes():
    lib = load_library()
    out = []
    for i in range(lib.wd_num_tiles()):
        shp = (ctypes.c_int * 4)()
        lib.wd_tile_shape(i, shp)
        out.append(tuple(shp))
    return out


def tile_infos():
    """[(BX,BY,BZ,BT, min_blocks_per_sm, has_fp32, has_fp64), ...] for every compiled launch configuration."""
    lib = load_library()
    out = []
    for i, shp in enumerate(tile_shapes()):
        info = (ctypes.c_int * 3)()
        lib.wd_tile_info(i, info)
        out.append(tuple(shp) + tuple(info))
    return out


def staging_rows():
    """[(16, BY, BZ, BT, stages, copies_ahead, min_blocks_per_sm, has_fp32, has_fp64), ...]: the compiled configurations of
    the stencil kernel with the shared-memory link pipeline (wd_set_link_staging)."""
    lib = load_library()
    out = []
    for i in range(lib.wd_num_staging_rows()):
        info = (ctypes.c_int * 9)()
        lib.wd_staging_row_info(i, info)
        out.append(tuple(info))
    return out


def _torch():
    import torch

    return torch


def cg_solve_host_queue(ctxs, systems, kappa, r_min, max_iter, outs):
    """A queue of host-buffer solves pipelined over two contexts (include/wilson_cg.h, cg_solve_host_begin / _run / _wait): the
    uploads of solve i+1 and the download of solve i-1 run while the GPU iterates on solve i.  `ctxs`: two WilsonContexts of
    the same lattice on two different streams; `systems`: a sequence of (U_host or None, eta_host); `outs[i]`: the pinned
    host buffer solve i writes (a buffer may be reused two solves later).  Returns the info dicts in order; every output is
    complete on return.  Argument marshalling only: the choreography of the header's example, nothing else."""
    if len(ctxs) != 2 or ctxs[0] is ctxs[1]:
        raise ValueError("two distinct contexts are needed")
    n = len(systems)
    infos = []
    if n == 0:
        return infos
    ctxs[0].cg_solve_host_begin(*systems[0])
    for i in range(n):
        if i + 1 < n:
            ctxs[(i + 1) % 2].cg_solve_host_begin(*systems[i + 1])
        infos.append(ctxs[i % 2].cg_solve_host_run(kappa, r_min, max_iter, outs[i]))
        if i > 0:
            ctxs[(i - 1) % 2].cg_solve_host_wait()
    ctxs[(n - 1) % 2].cg_solve_host_wait()
    return infos


def wd_noalloc_max_sites(precision: int) -> int:
    """Largest number of sites wd_norm2_noalloc accepts (its scratch is a static device array); needs no GPU."""
    return int(load_library().wd_noalloc_max_sites(int(precision)))


def wd_noalloc_prepare() -> None:
    """One-time set-up of wd_norm2_noalloc for the current device (e.g. before a stream capture begins)."""
    lib = load_library()
    rc = lib.wd_noalloc_prepare()
    if rc != 0:
        raise WilsonError(rc, lib.wd_noalloc_last_error().decode())


def wd_norm2_noalloc(a_native, n_sites: int, precision: int, out, stream=None) -> None:
    """<a,a> of a native spinor field without a context and without any allocation inside the library: enqueues the work on
    `stream` (a torch.cuda.Stream; None = the legacy default stream) and returns.  `out` is a CUDA float64 tensor of one
    element owned by the caller; read it after synchronising the stream.  Calls that overlap on the GPU race on the
    library's static scratch (include/wilson_cg.h)."""
    torch = _torch()
    lib = load_library()
    if not (isinstance(out, torch.Tensor) and out.is_cuda and out.dtype == torch.float64 and out.numel() >= 1):
        raise ValueError("out must be a CUDA float64 tensor with one element")
    sp = ctypes.c_void_p(stream.cuda_stream) if stream is not None else None
    rc = lib.wd_norm2_noalloc(int(precision), int(n_sites), ctypes.c_void_p(a_native.data_ptr()),
                              ctypes.c_void_p(out.data_ptr()), sp)
    if rc != 0:
        raise WilsonError(rc, lib.wd_noalloc_last_error().decode())


class WilsonContext:
    """wd_create / wd_destroy plus one method per ABI call.  Tensors are torch CUDA tensors
    (canonical layout: complex64/complex128 of shape (V,4,3,3) and (V,4,3); native buffers are opaque
    1-D real tensors from `empty_gauge()` / `empty_spinor()`)."""

    def __init__(self, dims, precision=32, bc_t=-1, stream=None):
        torch = _torch()
        if not torch.cuda.is_available():
            raise RuntimeError("wilson_cg needs a CUDA device (no CPU fallback)")
        self.lib = load_library()
        self.dims = tuple(int(d) for d in dims)
        self.volume = int(np.prod(self.dims))
        self.precision = int(precision)
        self.bc_t = int(bc_t)
        self.real_dtype = torch.float32 if precision == 32 else torch.float64
        self.complex_dtype = torch.complex64 if precision == 32 else torch.complex128
        self.np_complex = np.complex64 if precision == 32 else np.complex128
        self.stream = stream if stream is not None else torch.cuda.current_stream()
        self._ctx = ctypes.c_void_p()
        d = (ctypes.c_int * 4)(*self.dims)
        rc = self.lib.wd_create(ctypes.byref(self._ctx), d, self.precision, self.bc_t,
                                ctypes.c_void_p(self.stream.cuda_stream))
        if rc != WD_OK:
            raise WilsonError(rc, self.lib.wd_last_error(None).decode())

    # -- plumbing
    def close(self):
        if getattr(self, "_ctx", None) is not None and self._ctx.value:
            self.lib.wd_destroy(self._ctx)
            self._ctx = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def _check(self, rc, allow_not_converged=False):
        if rc == WD_OK or (allow_not_converged and rc in (WD_NOT_CONVERGED, WD_BREAKDOWN)):
            return rc
        raise WilsonError(rc, self.lib.wd_last_error(self._ctx).decode())

    @staticmethod
    def _p(t):
        return ctypes.c_void_p(t.data_ptr())

    def empty_gauge(self):
        torch = _torch()
        n = self.lib.wd_gauge_native_bytes(self._ctx) // (4 if self.precision == 32 else 8)
        return torch.empty(n, dtype=self.real_dtype, device="cuda")

    def empty_spinor(self):
        torch = _torch()
        n = self.lib.wd_spinor_native_bytes(self._ctx) // (4 if self.precision == 32 else 8)
        return torch.empty(n, dtype=self.real_dtype, device="cuda")

    def _canon(self, t, shape):
        torch = _torch()
        if t.dtype != self.complex_dtype or tuple(t.shape) != shape or not t.is_cuda or not t.is_contiguous():
            raise ValueError(f"expected contiguous CUDA {self.complex_dtype} tensor of shape {shape}")
        return t

    # -- a0
    def wd_pack_gauge(self, U_canonical, out=None):
        U_canonical = self._canon(U_canonical, (self.volume, 4, 3, 3))
        out = self.empty_gauge() if out is None else out
        self._check(self.lib.wd_pack_gauge(self._ctx, self._p(U_canonical), self._p(out)))
        return out

    def wd_pack_spinor(self, psi_canonical, out=None):
        psi_canonical = self._canon(psi_canonical, (self.volume, 4, 3))
        out = self.empty_spinor() if out is None else out
        self._check(self.lib.wd_pack_spinor(self._ctx, self._p(psi_canonical), self._p(out)))
        return out

    def wd_unpack_spinor(self, psi_native, out=None):
        torch = _torch()
        if out is None:
            out = torch.empty((self.volume, 4, 3), dtype=self.complex_dtype, device="cuda")
        self._check(self.lib.wd_unpack_spinor(self._ctx, self._p(psi_native), self._p(out)))
        return out

    # -- a7
    def wd_apply(self, U_native, psi_native, kappa, dagger=False, out=None):
        out = self.empty_spinor() if out is None else out
        self._check(self.lib.wd_apply(self._ctx, self._p(U_native), self._p(psi_native), self._p(out),
                                      float(kappa), int(bool(dagger))))
        return out

    def wd_apply_repeat(self, U_native, psi_native, kappa, dagger=False, reps=100, out=None):
        """device milliseconds per application over `reps` back-to-back applications enqueued from C"""
        out = self.empty_spinor() if out is None else out
        ms = ctypes.c_double()
        self._check(self.lib.wd_apply_repeat(self._ctx, self._p(U_native), self._p(psi_native), self._p(out),
                                             float(kappa), int(bool(dagger)), int(reps), ctypes.byref(ms)))
        return ms.value

    # -- a1..a6
    def cg_solve(self, U_native, eta_native, kappa, r_min, max_iter, out=None):
        out = self.empty_spinor() if out is None else out
        info = WdCgInfo()
        rc = self.lib.cg_solve(self._ctx, self._p(U_native), self._p(eta_native), self._p(out), float(kappa),
                               float(r_min), int(max_iter), ctypes.byref(info))
        self._check(rc, allow_not_converged=True)
        d = info.as_dict()
        d["status"] = rc
        return out, d

    # -- f4
    def bicgstab_solve(self, U_native, eta_native, kappa, r_min, max_iter, out=None):
        out = self.empty_spinor() if out is None else out
        info = WdCgInfo()
        rc = self.lib.bicgstab_solve(self._ctx, self._p(U_native), self._p(eta_native), self._p(out), float(kappa),
                                     float(r_min), int(max_iter), ctypes.byref(info))
        self._check(rc, allow_not_converged=True)
        d = info.as_dict()
        d["status"] = rc
        return out, d

    def wd_get_profile_bicgstab(self):
        ms = (ctypes.c_double * 5)()
        n = ctypes.c_long()
        self._check(self.lib.wd_get_profile_bicgstab(self._ctx, ms, ctypes.byref(n)))
        return {"ms": list(ms), "iterations": n.value}

    # -- f3: even-odd preconditioned CG
    def empty_eo_spinor(self):
        torch = _torch()
        n = self.lib.wd_eo_spinor_bytes(self._ctx) // (4 if self.precision == 32 else 8)
        return torch.empty(n, dtype=self.real_dtype, device="cuda")

    def empty_eo_gauge(self):
        torch = _torch()
        n = self.lib.wd_eo_gauge_bytes(self._ctx) // (4 if self.precision == 32 else 8)
        return torch.empty(n, dtype=self.real_dtype, device="cuda")

    def wd_eo_pack_spinor(self, psi_canonical, out=None):
        psi_canonical = self._canon(psi_canonical, (self.volume, 4, 3))
        out = self.empty_eo_spinor() if out is None else out
        self._check(self.lib.wd_eo_pack_spinor(self._ctx, self._p(psi_canonical), self._p(out)))
        return out

    def wd_eo_unpack_spinor(self, psi_eo, out=None):
        torch = _torch()
        if out is None:
            out = torch.empty((self.volume, 4, 3), dtype=self.complex_dtype, device="cuda")
        self._check(self.lib.wd_eo_unpack_spinor(self._ctx, self._p(psi_eo), self._p(out)))
        return out

    def wd_eo_pack_gauge(self, U_canonical, out=None):
        U_canonical = self._canon(U_canonical, (self.volume, 4, 3, 3))
        out = self.empty_eo_gauge() if out is None else out
        self._check(self.lib.wd_eo_pack_gauge(self._ctx, self._p(U_canonical), self._p(out)))
        return out

    def wd_eo_hop(self, U_eo, in_eo, out_eo, out_parity, dagger=False):
        self._check(self.lib.wd_eo_hop(self._ctx, self._p(U_eo), self._p(in_eo), self._p(out_eo), int(out_parity),
                                       int(bool(dagger))))
        return out_eo

    def cg_solve_eo(self, U_eo, eta_eo, kappa, r_min, max_iter, out=None):
        out = self.empty_eo_spinor() if out is None else out
        info = WdCgInfo()
        rc = self.lib.cg_solve_eo(self._ctx, self._p(U_eo), self._p(eta_eo), self._p(out), float(kappa),
                                  float(r_min), int(max_iter), ctypes.byref(info))
        self._check(rc, allow_not_converged=True)
        d = info.as_dict()
        d["status"] = rc
        return out, d

    def bicgstab_solve_eo(self, U_eo, eta_eo, kappa, r_min, max_iter, out=None):
        """even-odd preconditioned BiCGSTAB (BiCGSTAB on the Schur operator Mhat); status 2 = breakdown"""
        out = self.empty_eo_spinor() if out is None else out
        info = WdCgInfo()
        rc = self.lib.bicgstab_solve_eo(self._ctx, self._p(U_eo), self._p(eta_eo), self._p(out), float(kappa),
                                        float(r_min), int(max_iter), ctypes.byref(info))
        self._check(rc, allow_not_converged=True)
        d = info.as_dict()
        d["status"] = rc
        return out, d

    def wd_get_profile_eo_bicgstab(self):
        ms = (ctypes.c_double * 7)()
        n = ctypes.c_long()
        self._check(self.lib.wd_get_profile_eo_bicgstab(self._ctx, ms, ctypes.byref(n)))
        return {"ms": list(ms), "iterations": n.value}

    # -- f3: several right-hand sides at once (fields: (nrhs, n) real tensors, row j = native spinor of source j)
    def empty_multi_spinor(self, nrhs):
        torch = _torch()
        n = self.lib.wd_spinor_native_bytes(self._ctx) // (4 if self.precision == 32 else 8)
        return torch.empty((int(nrhs), n), dtype=self.real_dtype, device="cuda")

    def wd_apply_multi(self, U_native, in_multi, kappa, dagger=False, out=None):
        nrhs = in_multi.shape[0]
        out = self.empty_multi_spinor(nrhs) if out is None else out
        self._check(self.lib.wd_apply_multi(self._ctx, self._p(U_native), self._p(in_multi), self._p(out), int(nrhs),
                                            float(kappa), int(bool(dagger))))
        return out

    def cg_solve_multi(self, U_native, eta_multi, kappa, r_min, max_iter, out=None):
        nrhs = eta_multi.shape[0]
        out = self.empty_multi_spinor(nrhs) if out is None else out
        infos = (WdCgInfo * nrhs)()
        rc = self.lib.cg_solve_multi(self._ctx, self._p(U_native), self._p(eta_multi), self._p(out), int(nrhs),
                                     float(kappa), float(r_min), int(max_iter), infos)
        self._check(rc, allow_not_converged=True)
        return out, [dict(i.as_dict(), status=0 if i.converged else 1) for i in infos]

    # -- f2: the paper's coordinate-format route
    def wd_coo_nnz(self):
        return int(self.lib.wd_coo_nnz(self._ctx))

    def wd_coo_assemble(self, U_native, kappa, dagger=False):
        """(val complex[nnz], row int32[nnz], col int32[nnz]) CUDA tensors"""
        torch = _torch()
        nnz = self.wd_coo_nnz()
        val = torch.empty(nnz, dtype=self.complex_dtype, device="cuda")
        row = torch.empty(nnz, dtype=torch.int32, device="cuda")
        col = torch.empty(nnz, dtype=torch.int32, device="cuda")
        self._check(self.lib.wd_coo_assemble(self._ctx, self._p(U_native), float(kappa), int(bool(dagger)),
                                             self._p(val), self._p(row), self._p(col)))
        return val, row, col

    def wd_coo_spmv(self, val, row, col, vec_canonical, out=None):
        torch = _torch()
        vec_canonical = self._canon(vec_canonical, (self.volume, 4, 3))
        if val.dtype != self.complex_dtype or row.dtype != torch.int32 or col.dtype != torch.int32:
            raise ValueError("val must have the ctx complex dtype, row/col int32")
        if not (val.is_cuda and row.is_cuda and col.is_cuda) or not (row.numel() == col.numel() == val.numel()):
            raise ValueError("val, row, col must be CUDA tensors of equal length")
        out = torch.empty_like(vec_canonical) if out is None else out
        self._check(self.lib.wd_coo_spmv(self._ctx, val.numel(), self._p(val), self._p(row), self._p(col),
                                         self._p(vec_canonical), self._p(out)))
        return out

    def wd_cg_history(self, n=None):
        n = int(n) if n is not None else 1 << 20
        buf = np.zeros(n, dtype=np.float64)
        got = self.lib.wd_cg_history(self._ctx, buf.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), n)
        if got < 0:
            self._check(got)
        return buf[:got].copy()

    def wd_norm2(self, a_native):
        res = ctypes.c_double()
        self._check(self.lib.wd_norm2(self._ctx, self._p(a_native), ctypes.byref(res)))
        return res.value

    # -- host-buffer forms (numpy arrays or pinned torch CPU tensors, canonical layout)
    def _host_ptr(self, a, shape, writable=False):
        torch = _torch()
        if isinstance(a, torch.Tensor):
            if a.is_cuda or a.dtype != self.complex_dtype or tuple(a.shape) != shape or not a.is_contiguous():
                raise ValueError(f"expected contiguous CPU {self.complex_dtype} tensor of shape {shape}")
            return ctypes.c_void_p(a.data_ptr())
        if a.dtype != self.np_complex or a.shape != shape or not a.flags.c_contiguous:
            raise ValueError(f"expected C-contiguous {self.np_complex} array of shape {shape}")
        if writable and not a.flags.writeable:
            raise ValueError("output array is read-only")
        return ctypes.c_void_p(a.ctypes.data)

    def wd_apply_host(self, U_host, psi_host, kappa, dagger=False, out=None):
        V = self.volume
        out = np.empty((V, 4, 3), dtype=self.np_complex) if out is None else out
        up = self._host_ptr(U_host, (V, 4, 3, 3)) if U_host is not None else None
        self._check(self.lib.wd_apply_host(self._ctx, up, self._host_ptr(psi_host, (V, 4, 3)),
                                           self._host_ptr(out, (V, 4, 3), True), float(kappa), int(bool(dagger))))
        return out

    def cg_solve_host(self, U_host, eta_host, kappa, r_min, max_iter, out=None):
        V = self.volume
        out = np.empty((V, 4, 3), dtype=self.np_complex) if out is None else out
        up = self._host_ptr(U_host, (V, 4, 3, 3)) if U_host is not None else None
        info = WdCgInfo()
        rc = self.lib.cg_solve_host(self._ctx, up, self._host_ptr(eta_host, (V, 4, 3)),
                                    self._host_ptr(out, (V, 4, 3), True), float(kappa), float(r_min),
                                    int(max_iter), ctypes.byref(info))
        self._check(rc, allow_not_converged=True)
        d = info.as_dict()
        d["status"] = rc
        return out, d

    # -- split-phase form: with two contexts the transfers of one solve overlap the iterations of another
    def cg_solve_host_begin(self, U_host, eta_host):
        """enqueue the uploads of U_host (None = the gauge field already on this ctx) and eta_host; returns at once.  The
        buffers (pinned, canonical layout) must stay untouched until cg_solve_host_run on this ctx has returned."""
        V = self.volume
        up = self._host_ptr(U_host, (V, 4, 3, 3)) if U_host is not None else None
        self._check(self.lib.cg_solve_host_begin(self._ctx, up, self._host_ptr(eta_host, (V, 4, 3))))

    def cg_solve_host_run(self, kappa, r_min, max_iter, out):
        """the solve on the staged fields; enqueues the download into `out` (complete after cg_solve_host_wait)"""
        info = WdCgInfo()
        rc = self.lib.cg_solve_host_run(self._ctx, self._host_ptr(out, (self.volume, 4, 3), True), float(kappa),
                                        float(r_min), int(max_iter), ctypes.byref(info))
        self._check(rc, allow_not_converged=True)
        d = info.as_dict()
        d["status"] = rc
        return d

    def cg_solve_host_wait(self):
        self._check(self.lib.cg_solve_host_wait(self._ctx))

    # -- tuning knobs
    def wd_set_tile(self, index):
        self._check(self.lib.wd_set_tile(self._ctx, int(index)))

    def wd_get_tile(self):
        return int(self.lib.wd_get_tile(self._ctx))

    def wd_set_profile(self, on):
        """False/0 off, True/1 time the kernels of every iteration, n > 1 of every n-th iteration (cg_solve only)"""
        self._check(self.lib.wd_set_profile(self._ctx, int(on)))

    def wd_get_profile(self):
        """{'a2_ms', 'a3_ms', 'a4_ms', 'iterations'}: accumulated device time per kernel class of the CG loop."""
        ms = (ctypes.c_double * 3)()
        n = ctypes.c_long()
        self._check(self.lib.wd_get_profile(self._ctx, ms, ctypes.byref(n)))
        return {"a2_ms": ms[0], "a3_ms": ms[1], "a4_ms": ms[2], "iterations": n.value}

    def wd_set_cg_mode(self, mode):
        """0 automatic, 1 three kernels per iteration, 2 whole solve in one cooperative launch (thread per site), 6 one launch with
        the hopping sum split over four warps, 9 one launch with the lattice resident in the shared memory of a cluster, 10 one launch with the gauge field resident in
        shared memory"""
        self._check(self.lib.wd_set_cg_mode(self._ctx, int(mode)))

    def wd_set_gauge_recon(self, reals_per_link):
        """18 (default) or 12 reals stored per link; call before wd_pack_gauge / empty_gauge"""
        self._check(self.lib.wd_set_gauge_recon(self._ctx, int(reals_per_link)))

    def wd_get_gauge_recon(self):
        return int(self.lib.wd_get_gauge_recon(self._ctx))

    def wd_set_zchunk(self, layers):
        self._check(self.lib.wd_set_zchunk(self._ctx, int(layers)))

    def wd_set_small_tile(self, index):
        self._check(self.lib.wd_set_small_tile(self._ctx, int(index)))

    def wd_set_coo_fast(self, on):
        """1 (default): wd_coo_spmv uses the sorted-row kernel for the arrays wd_coo_assemble wrote; 0: always the any-order kernel"""
        self._check(self.lib.wd_set_coo_fast(self._ctx, int(on)))

    def wd_set_link_staging(self, row):
        """row of staging_rows() for the stencil passes of wd_apply / cg_solve (three-kernel driver); -1 = off"""
        self._check(self.lib.wd_set_link_staging(self._ctx, int(row)))

    def wd_get_link_staging(self):
        return int(self.lib.wd_get_link_staging(self._ctx))

    def wd_set_poll_interval(self, n):
        self._check(self.lib.wd_set_poll_interval(self._ctx, int(n)))
