"""Seeded synthetic lattices: gauge links, sources, gauge transforms (numpy only).

This module is the ONE piece shared by the CPU oracle (`oracle/`) and the CUDA path:
it produces inputs and holds none of the method's arithmetic (no Wilson operator, no
CG, no gamma matrices).  It never imports the CUDA binding or the oracle.

What it stands in for: the paper does not say which gauge fields or sources it ran on
(PAPER.md:44 gives only the volumes 4^4..14^4; PAPER.md:32 quotes 48^3x96).  The five
workloads are those of BASELINE.json `configs`; the recipe is SURVEY.md §8(d) and
DESIGN.md "Input recipe":

* RNG: numpy Generator(PCG64) seeded from SeedSequence([BASE_SEED, cfg, field, t]) — one
  stream per (config, field, t-slice), so generation is slice-by-slice and independent
  of chunking.  Values are drawn in canonical-layout order within a slice, real part
  then imaginary part of each complex number.
* Complex Gaussian: re and im each ~ N(0,1), independent (reading G11).
* Haar SU(3) (configs 0, 2): Z complex Gaussian 3x3, Z = QR, Q <- Q diag(R_ii/|R_ii|)
  (i.e. the QR factor with positive diagonal R = Gram-Schmidt on the columns of Z), then
  Q <- Q exp(-i arg(det Q)/3) (principal branch) so det = 1 (reading G12).
* Near-identity SU(3) (configs 1, 3, 4): A = (Z - Z^H)/2, M = 1 + eps A, eps = 0.3,
  projected by the same Gram-Schmidt + determinant-phase routine (reading G13).

Canonical layouts (the C-ABI's caller-visible layouts, include/wilson_cg.h):
  site s = x + Lx (y + Ly (z + Lz t));  U[s][mu][a][b];  psi[s][alpha][a].
"""
from __future__ import annotations

from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass
import os

import numpy as np

BASE_SEED = 211114958

FIELD_GAUGE = 0
FIELD_SOURCE = 1
FIELD_GAUGE_TRANSFORM = 2
FIELD_AUX = 3  # extra test vectors (chi, random psi) for parity/property tests


@dataclass(frozen=True)
class LatticeConfig:
    """One BASELINE.json workload.  dims = (Lx, Ly, Lz, Lt)."""

    index: int
    name: str
    dims: tuple
    kappa: float
    links: str  # "haar" | "near_identity" | "unit"
    r_min: float
    max_iter: int
    eps: float = 0.3
    bc_t: int = -1  # antiperiodic in t

    @property
    def volume(self) -> int:
        lx, ly, lz, lt = self.dims
        return lx * ly * lz * lt


CONFIGS = (
    LatticeConfig(0, "4^4", (4, 4, 4, 4), 0.12, "haar", 1e-6, 1000),
    LatticeConfig(1, "8^4", (8, 8, 8, 8), 0.124, "near_identity", 1e-6, 1000),
    LatticeConfig(2, "14^4", (14, 14, 14, 14), 0.12, "haar", 1e-6, 1000),
    LatticeConfig(3, "32^4", (32, 32, 32, 32), 0.1245, "near_identity", 1e-6, 5000),
    LatticeConfig(4, "48^3x96", (48, 48, 48, 96), 0.124, "near_identity", 1e-6, 5000),
)


def slice_rng(cfg: int, field: int, t: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(np.random.SeedSequence([BASE_SEED, cfg, field, t])))


def complex_gaussian(rng: np.random.Generator, shape) -> np.ndarray:
    """re, im each N(0,1); drawn as (..., 2) so re comes before im for each element."""
    z = rng.standard_normal(tuple(shape) + (2,))
    return z[..., 0] + 1j * z[..., 1]


def project_su3(m: np.ndarray) -> np.ndarray:
    """Batched (..., 3, 3) -> SU(3): Gram-Schmidt on columns (== QR with positive diag R),
    then remove the determinant phase with the principal cube root."""
    c0 = m[..., :, 0]
    c1 = m[..., :, 1]
    c2 = m[..., :, 2]
    q0 = c0 / np.linalg.norm(c0, axis=-1, keepdims=True)
    c1 = c1 - q0 * np.sum(np.conj(q0) * c1, axis=-1, keepdims=True)
    q1 = c1 / np.linalg.norm(c1, axis=-1, keepdims=True)
    c2 = c2 - q0 * np.sum(np.conj(q0) * c2, axis=-1, keepdims=True)
    c2 = c2 - q1 * np.sum(np.conj(q1) * c2, axis=-1, keepdims=True)
    q2 = c2 / np.linalg.norm(c2, axis=-1, keepdims=True)
    q = np.stack([q0, q1, q2], axis=-1)
    det = (
        q[..., 0, 0] * (q[..., 1, 1] * q[..., 2, 2] - q[..., 1, 2] * q[..., 2, 1])
        - q[..., 0, 1] * (q[..., 1, 0] * q[..., 2, 2] - q[..., 1, 2] * q[..., 2, 0])
        + q[..., 0, 2] * (q[..., 1, 0] * q[..., 2, 1] - q[..., 1, 1] * q[..., 2, 0])
    )
    phase = np.exp(-1j * np.angle(det) / 3.0)
    return q * phase[..., None, None]


def _links_from_gaussian(z: np.ndarray, links: str, eps: float) -> np.ndarray:
    if links == "haar":
        return project_su3(z)
    if links == "near_identity":
        a = 0.5 * (z - np.conj(np.swapaxes(z, -1, -2)))
        return project_su3(np.eye(3) + eps * a)
    raise ValueError(f"unknown link family {links!r}")


def gauge_slice(cfg: int, dims, t: int, links: str, eps: float = 0.3) -> np.ndarray:
    """Links of t-slice t: complex128 array (Lx*Ly*Lz, 4, 3, 3), x fastest."""
    lx, ly, lz, _ = dims
    n = lx * ly * lz
    if links == "unit":
        out = np.zeros((n, 4, 3, 3), dtype=np.complex128)
        out[..., 0, 0] = out[..., 1, 1] = out[..., 2, 2] = 1.0
        return out
    z = complex_gaussian(slice_rng(cfg, FIELD_GAUGE, t), (n, 4, 3, 3))
    return _links_from_gaussian(z, links, eps)


def source_slice(cfg: int, dims, t: int, field: int = FIELD_SOURCE) -> np.ndarray:
    """Gaussian spinor on t-slice t: complex128 (Lx*Ly*Lz, 4, 3)."""
    lx, ly, lz, _ = dims
    return complex_gaussian(slice_rng(cfg, field, t), (lx * ly * lz, 4, 3))


def _assemble(dims, tail_shape, dtype, make_slice, workers=None) -> np.ndarray:
    lx, ly, lz, lt = dims
    n = lx * ly * lz
    out = np.empty((n * lt,) + tail_shape, dtype=dtype)

    def fill(t):
        out[t * n:(t + 1) * n] = make_slice(t)

    workers = workers or min(lt, os.cpu_count() or 1, 16)
    if workers <= 1 or n * lt < 1 << 16:
        for t in range(lt):
            fill(t)
    else:
        with ThreadPoolExecutor(workers) as pool:
            list(pool.map(fill, range(lt)))
    return out


def gauge_field(cfg: int, dims, links: str, eps: float = 0.3, dtype=np.complex128) -> np.ndarray:
    """Canonical gauge field U[s][mu][a][b], shape (V, 4, 3, 3).  `dtype` complex64 gives the
    fp32-rounded field (generated in fp64, rounded once)."""
    return _assemble(dims, (4, 3, 3), dtype, lambda t: gauge_slice(cfg, dims, t, links, eps))


def source_field(cfg: int, dims, dtype=np.complex128, field: int = FIELD_SOURCE) -> np.ndarray:
    """Canonical Gaussian spinor eta[s][alpha][a], shape (V, 4, 3)."""
    return _assemble(dims, (4, 3), dtype, lambda t: source_slice(cfg, dims, t, field))


def gauge_transform_field(cfg: int, dims) -> np.ndarray:
    """Haar SU(3) matrix g(x) per site, shape (V, 3, 3) — used by the covariance pins."""
    lx, ly, lz, _ = dims
    n = lx * ly * lz
    return _assemble(
        dims, (3, 3), np.complex128,
        lambda t: project_su3(complex_gaussian(slice_rng(cfg, FIELD_GAUGE_TRANSFORM, t), (n, 3, 3))))


def config_inputs(cfg: LatticeConfig, dtype=np.complex128):
    """(U, eta) of a BASELINE.json config in canonical layout."""
    u = gauge_field(cfg.index, cfg.dims, cfg.links, cfg.eps, dtype=dtype)
    eta = source_field(cfg.index, cfg.dims, dtype=dtype)
    return u, eta
