"""ctypes front end of the fp64 CPU oracle (oracle/wilson_oracle.c) — TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this.  It does not import the CUDA package and the CUDA package does not import it.
All arithmetic lives in wilson_oracle.c (see its header for citations and pins); this file
only compiles it with gcc and marshals numpy arrays.

Canonical layouts: U complex128 (V, 4, 3, 3), psi complex128 (V, 4, 3), site index
s = x + Lx (y + Ly (z + Lz t)), dims = (Lx, Ly, Lz, Lt).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "wilson_oracle.c")
_LIB = os.path.join(_HERE, "libwilson_oracle.so")
_lock = threading.Lock()
_lib = None


class OracleCgInfo(ctypes.Structure):
    _fields_ = [
        ("iterations", ctypes.c_int),
        ("converged", ctypes.c_int),
        ("rel_residual", ctypes.c_double),
        ("eta_norm2", ctypes.c_double),
        ("seconds", ctypes.c_double),
    ]


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2 -fopenmp).  Returns the path of the shared object."""
    with _lock:
        if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
            tmp = _LIB + f".{os.getpid()}.tmp"
            subprocess.check_call(
                ["gcc", "-std=c99", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"])
            os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        i4 = ctypes.POINTER(ctypes.c_int)
        dp = ctypes.POINTER(ctypes.c_double)
        lib.oracle_wd_apply.argtypes = [i4, ctypes.c_int, dp, dp, dp, ctypes.c_double, ctypes.c_int]
        lib.oracle_wd_apply.restype = ctypes.c_int
        lib.oracle_wd_apply_sites.argtypes = [i4, ctypes.c_int, dp, dp, dp, ctypes.c_double, ctypes.c_int,
                                              ctypes.POINTER(ctypes.c_long), ctypes.c_long]
        lib.oracle_wd_apply_sites.restype = ctypes.c_int
        lib.oracle_cg_solve.argtypes = [i4, ctypes.c_int, dp, dp, dp, ctypes.c_double, ctypes.c_double,
                                        ctypes.c_int, ctypes.POINTER(OracleCgInfo), dp]
        lib.oracle_cg_solve.restype = ctypes.c_int
        lib.oracle_bicgstab_solve.argtypes = lib.oracle_cg_solve.argtypes
        lib.oracle_bicgstab_solve.restype = ctypes.c_int
        ip = ctypes.POINTER(ctypes.c_int)
        lib.oracle_coo_nnz.argtypes = [i4]
        lib.oracle_coo_nnz.restype = ctypes.c_long
        lib.oracle_coo_assemble.argtypes = [i4, ctypes.c_int, dp, ctypes.c_double, ctypes.c_int, dp, ip, ip]
        lib.oracle_coo_assemble.restype = ctypes.c_int
        lib.oracle_coo_spmv.argtypes = [ctypes.c_long, dp, ip, ip, dp, dp, ctypes.c_long]
        lib.oracle_coo_spmv.restype = ctypes.c_int
        lib.oracle_cg_solve_eo.argtypes = lib.oracle_cg_solve.argtypes
        lib.oracle_cg_solve_eo.restype = ctypes.c_int
        lib.oracle_bicgstab_solve_eo.argtypes = lib.oracle_cg_solve.argtypes
        lib.oracle_bicgstab_solve_eo.restype = ctypes.c_int
        lib.oracle_schur_apply.argtypes = lib.oracle_wd_apply.argtypes
        lib.oracle_schur_apply.restype = ctypes.c_int
        lib.oracle_norm2.argtypes = [dp, ctypes.c_long]
        lib.oracle_norm2.restype = ctypes.c_double
        lib.oracle_num_threads.restype = ctypes.c_int
        lib.oracle_set_num_threads.argtypes = [ctypes.c_int]
        _lib = lib
    return _lib


def _dims(dims):
    d = (ctypes.c_int * 4)(*[int(v) for v in dims])
    vol = int(dims[0]) * int(dims[1]) * int(dims[2]) * int(dims[3])
    return d, vol


def _c128(a, shape):
    a = np.ascontiguousarray(a, dtype=np.complex128)
    if a.shape != shape:
        raise ValueError(f"expected shape {shape}, got {a.shape}")
    return a


def _ptr(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def wd_apply(dims, U, psi, kappa, dagger=False, bc_t=-1):
    """D psi (dagger False) or D-dagger psi on the whole lattice (reading C-1)."""
    d, vol = _dims(dims)
    U = _c128(U, (vol, 4, 3, 3))
    psi = _c128(psi, (vol, 4, 3))
    out = np.empty_like(psi)
    rc = _load().oracle_wd_apply(d, int(bc_t), _ptr(U), _ptr(psi), _ptr(out), float(kappa), int(bool(dagger)))
    if rc != 0:
        raise RuntimeError(f"oracle_wd_apply failed: {rc}")
    return out


def wd_apply_sites(dims, U, psi, kappa, sites, dagger=False, bc_t=-1):
    """The same operator evaluated at the listed site indices only: returns (n, 4, 3)."""
    d, vol = _dims(dims)
    U = _c128(U, (vol, 4, 3, 3))
    psi = _c128(psi, (vol, 4, 3))
    sites = np.ascontiguousarray(sites, dtype=np.int64)
    out = np.empty((sites.size, 4, 3), dtype=np.complex128)
    rc = _load().oracle_wd_apply_sites(
        d, int(bc_t), _ptr(U), _ptr(psi), _ptr(out), float(kappa), int(bool(dagger)),
        sites.ctypes.data_as(ctypes.POINTER(ctypes.c_long)), sites.size)
    if rc != 0:
        raise RuntimeError(f"oracle_wd_apply_sites failed: {rc}")
    return out


def cg_solve(dims, U, eta, kappa, r_min, max_iter, bc_t=-1, history=False):
    """The paper's CG on D D-dagger, then psi = D-dagger y (readings G1-G5).

    Returns (psi, info dict).  info: iterations, converged, rel_residual (recursed), eta_norm2,
    seconds, status (0 converged / 1 max_iter), and rr_history if asked for."""
    d, vol = _dims(dims)
    U = _c128(U, (vol, 4, 3, 3))
    eta = _c128(eta, (vol, 4, 3))
    psi = np.empty_like(eta)
    info = OracleCgInfo()
    hist = np.zeros(max_iter + 1, dtype=np.float64) if history else None
    rc = _load().oracle_cg_solve(
        d, int(bc_t), _ptr(U), _ptr(eta), _ptr(psi), float(kappa), float(r_min), int(max_iter),
        ctypes.byref(info), _ptr(hist) if history else None)
    if rc < 0:
        raise RuntimeError(f"oracle_cg_solve failed: {rc}")
    out = {
        "iterations": info.iterations,
        "converged": bool(info.converged),
        "rel_residual": info.rel_residual,
        "eta_norm2": info.eta_norm2,
        "seconds": info.seconds,
        "status": rc,
    }
    if history:
        out["rr_history"] = hist[: info.iterations + 1].copy()
    return psi, out


def bicgstab_solve(dims, U, eta, kappa, r_min, max_iter, bc_t=-1, history=False):
    """BiCGSTAB on D directly (the paper names the method at PAPER.md:32; listing = reading B1).

    Returns (psi, info) like cg_solve; status 2 = breakdown."""
    d, vol = _dims(dims)
    U = _c128(U, (vol, 4, 3, 3))
    eta = _c128(eta, (vol, 4, 3))
    psi = np.empty_like(eta)
    info = OracleCgInfo()
    hist = np.zeros(max_iter + 1, dtype=np.float64) if history else None
    rc = _load().oracle_bicgstab_solve(
        d, int(bc_t), _ptr(U), _ptr(eta), _ptr(psi), float(kappa), float(r_min), int(max_iter),
        ctypes.byref(info), _ptr(hist) if history else None)
    if rc < 0:
        raise RuntimeError(f"oracle_bicgstab_solve failed: {rc}")
    out = {
        "iterations": info.iterations,
        "converged": bool(info.converged),
        "rel_residual": info.rel_residual,
        "eta_norm2": info.eta_norm2,
        "seconds": info.seconds,
        "status": rc,
    }
    if history:
        out["rr_history"] = hist[: info.iterations + 1].copy()
    return psi, out


def schur_apply(dims, U, v, kappa, dagger=False, bc_t=-1):
    """Mhat v_e = (1 - kappa^2 H_eo H_oe) v_e (or Mhat-dagger) on the even part of v; odd sites of the result are 0."""
    d, vol = _dims(dims)
    U = _c128(U, (vol, 4, 3, 3))
    v = _c128(v, (vol, 4, 3))
    out = np.empty_like(v)
    rc = _load().oracle_schur_apply(d, int(bc_t), _ptr(U), _ptr(v), _ptr(out), float(kappa), int(bool(dagger)))
    if rc != 0:
        raise RuntimeError(f"oracle_schur_apply failed: {rc}")
    return out


def cg_solve_eo(dims, U, eta, kappa, r_min, max_iter, bc_t=-1, history=False):
    """Even-odd preconditioned CG (reading E1): the paper's recurrence on Mhat Mhat-dagger, then
    psi_e = Mhat-dagger y and psi_o = eta_o + kappa H_oe psi_e.  Returns (psi, info) like cg_solve."""
    d, vol = _dims(dims)
    U = _c128(U, (vol, 4, 3, 3))
    eta = _c128(eta, (vol, 4, 3))
    psi = np.empty_like(eta)
    info = OracleCgInfo()
    hist = np.zeros(max_iter + 1, dtype=np.float64) if history else None
    rc = _load().oracle_cg_solve_eo(
        d, int(bc_t), _ptr(U), _ptr(eta), _ptr(psi), float(kappa), float(r_min), int(max_iter),
        ctypes.byref(info), _ptr(hist) if history else None)
    if rc < 0:
        raise RuntimeError(f"oracle_cg_solve_eo failed: {rc}")
    out = {
        "iterations": info.iterations,
        "converged": bool(info.converged),
        "rel_residual": info.rel_residual,
        "eta_norm2": info.eta_norm2,
        "seconds": info.seconds,
        "status": rc,
    }
    if history:
        out["rr_history"] = hist[: info.iterations + 1].copy()
    return psi, out


def bicgstab_solve_eo(dims, U, eta, kappa, r_min, max_iter, bc_t=-1, history=False):
    """Even-odd preconditioned BiCGSTAB (readings E1 + B1 composed = EB1): the BiCGSTAB listing on Mhat, then
    psi_o = eta_o + kappa H_oe psi_e.  Returns (psi, info) like cg_solve; status 2 = breakdown."""
    d, vol = _dims(dims)
    U = _c128(U, (vol, 4, 3, 3))
    eta = _c128(eta, (vol, 4, 3))
    psi = np.empty_like(eta)
    info = OracleCgInfo()
    hist = np.zeros(max_iter + 1, dtype=np.float64) if history else None
    rc = _load().oracle_bicgstab_solve_eo(
        d, int(bc_t), _ptr(U), _ptr(eta), _ptr(psi), float(kappa), float(r_min), int(max_iter),
        ctypes.byref(info), _ptr(hist) if history else None)
    if rc < 0:
        raise RuntimeError(f"oracle_bicgstab_solve_eo failed: {rc}")
    out = {
        "iterations": info.iterations,
        "converged": bool(info.converged),
        "rel_residual": info.rel_residual,
        "eta_norm2": info.eta_norm2,
        "seconds": info.seconds,
        "status": rc,
    }
    if history:
        out["rr_history"] = hist[: info.iterations + 1].copy()
    return psi, out


def coo_assemble(dims, U, kappa, dagger=False, bc_t=-1):
    """D (or D-dagger) in the paper's coordinate format: (val complex128[nnz], row int32[nnz],
    col int32[nnz]), nnz = 588 V, entry order as documented in wilson_oracle.c."""
    d, vol = _dims(dims)
    U = _c128(U, (vol, 4, 3, 3))
    nnz = int(_load().oracle_coo_nnz(d))
    val = np.empty(nnz, dtype=np.complex128)
    row = np.empty(nnz, dtype=np.int32)
    col = np.empty(nnz, dtype=np.int32)
    ip = ctypes.POINTER(ctypes.c_int)
    rc = _load().oracle_coo_assemble(d, int(bc_t), _ptr(U), float(kappa), int(bool(dagger)), _ptr(val),
                                     row.ctypes.data_as(ip), col.ctypes.data_as(ip))
    if rc != 0:
        raise RuntimeError(f"oracle_coo_assemble failed: {rc}")
    return val, row, col


def coo_spmv(val, row, col, vec):
    """The paper's SpMV loop out[Row[k]] += Val[k] * in[Col[k]], serial, fp64."""
    val = np.ascontiguousarray(val, dtype=np.complex128)
    row = np.ascontiguousarray(row, dtype=np.int32)
    col = np.ascontiguousarray(col, dtype=np.int32)
    shape = np.shape(vec)
    vin = np.ascontiguousarray(vec, dtype=np.complex128).reshape(-1)
    out = np.empty_like(vin)
    ip = ctypes.POINTER(ctypes.c_int)
    rc = _load().oracle_coo_spmv(val.size, _ptr(val), row.ctypes.data_as(ip), col.ctypes.data_as(ip), _ptr(vin),
                                 _ptr(out), out.size)
    if rc != 0:
        raise RuntimeError(f"oracle_coo_spmv failed: {rc}")
    return out.reshape(shape)


def norm2(a) -> float:
    a = np.ascontiguousarray(a, dtype=np.complex128)
    return float(_load().oracle_norm2(_ptr(a), a.size))


def true_residual(dims, U, eta, psi, kappa, bc_t=-1) -> float:
    """|eta - D psi| / |eta| with the oracle's fp64 D (reading G16)."""
    r = np.asarray(eta, dtype=np.complex128) - wd_apply(dims, U, psi, kappa, False, bc_t)
    return float(np.sqrt(norm2(r) / norm2(eta)))


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def set_num_threads(n: int) -> None:
    _load().oracle_set_num_threads(int(n))
