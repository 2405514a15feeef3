"""-m gpu parity tests of the SURVEY.md 8(f) rows built after the CG path: BiCGSTAB on D (f4), the paper's COO
SpMV (f2), 12-real link reconstruction (f3).  Same rules as test_gpu_parity.py: the CUDA path through the C ABI
against the fp64 CPU oracle on the same seeded inputs.

Tolerances:
  * bicgstab_solve: true residual |eta - D psi|/|eta| (oracle's fp64 D) <= 2x the oracle's and < 2 r_min; iteration
    count identical in fp64 and within max(1, 5 %) in fp32 (BiCGSTAB's omega steps amplify rounding differences;
    the CG's +-2 % of north_star is stated for the CG only);
  * COO: Row, Col bit-exact; Val and SpMV results to the fp32 / fp64 rounding of one product (1e-6 / 1e-14 relative).
"""
import math

import numpy as np
import pytest

from paper_2111_14958_b200 import inputs
import gpu_util as gu
import lattice_math as lm

pytestmark = pytest.mark.gpu
CFG_TEST = 800


@pytest.fixture(scope="module")
def wilson():
    import torch

    assert torch.cuda.is_available(), "the -m gpu tests need a CUDA device"
    from paper_2111_14958_b200 import build as wbuild
    from paper_2111_14958_b200 import wilson as w

    wbuild.build()
    w.load_library()
    return w


def bicgstab_on_gpu(ctx, U, eta, kappa, r_min, max_iter):
    Un = ctx.wd_pack_gauge(gu.to_device(U))
    en = ctx.wd_pack_spinor(gu.to_device(eta))
    psi_n, info = ctx.bicgstab_solve(Un, en, kappa, r_min, max_iter)
    return gu.to_host(ctx.wd_unpack_spinor(psi_n)), info


# ---------------------------------------------------------------- f4: BiCGSTAB
@pytest.mark.parametrize("precision,r_min", [(32, 1e-6), (64, 1e-10)])
@pytest.mark.parametrize("cfg_index", [0, 1, 2])
def test_bicgstab_baseline_configs(wilson, oracle, cfg_index, precision, r_min):
    cfg = inputs.CONFIGS[cfg_index]
    U, eta = gu.config_fields(cfg.index, precision)
    U64, eta64 = U.astype(np.complex128), eta.astype(np.complex128)
    with wilson.WilsonContext(cfg.dims, precision, cfg.bc_t) as ctx:
        psi, info = bicgstab_on_gpu(ctx, U, eta, cfg.kappa, r_min, cfg.max_iter)
        hist = ctx.wd_cg_history()
    psi_o, info_o = oracle.bicgstab_solve(cfg.dims, U64, eta64, cfg.kappa, r_min, cfg.max_iter, cfg.bc_t, history=True)
    assert info["status"] == 0 and info["converged"] == 1 and info["cg_mode"] == 3 and info_o["converged"]
    assert info["kernel_launches"] >= 5 * info["iterations"] + 1
    slack = 0 if precision == 64 else max(1, int(0.05 * info_o["iterations"] + 0.5))
    assert abs(info["iterations"] - info_o["iterations"]) <= slack, (info["iterations"], info_o["iterations"])
    res_gpu = oracle.true_residual(cfg.dims, U64, eta64, psi.astype(np.complex128), cfg.kappa, cfg.bc_t)
    res_orc = oracle.true_residual(cfg.dims, U64, eta64, psi_o, cfg.kappa, cfg.bc_t)
    assert res_gpu < 2.0 * r_min
    if info["iterations"] == info_o["iterations"]:
        assert res_gpu <= 2.0 * res_orc, (res_gpu, res_orc)
    assert len(hist) == info["iterations"] + 1
    n = min(len(hist), len(info_o["rr_history"]))
    rel = np.abs(hist[:n] - info_o["rr_history"][:n]) / info_o["rr_history"][:n]
    assert rel[0] < (1e-6 if precision == 32 else 1e-13)
    assert np.max(rel[: max(2, n // 2)]) < (5e-2 if precision == 32 else 1e-6), rel
    diff = np.linalg.norm(psi - psi_o) / np.linalg.norm(psi_o)
    assert diff < 4.0 * r_min / (1.0 - 8.0 * cfg.kappa) * (1 + 8 * cfg.kappa)


@pytest.mark.parametrize("precision", [32, 64])
def test_bicgstab_ragged_lattice_and_cg_agree(wilson, oracle, precision):
    """5x7x4x6 (volume not a multiple of the 16-site block: pad lanes) and both solvers give the same psi"""
    dims, kappa = (5, 7, 4, 6), 0.12
    cdt = gu.np_complex(precision)
    U = inputs.gauge_field(CFG_TEST + 1, dims, "haar", dtype=cdt)
    eta = inputs.source_field(CFG_TEST + 1, dims, dtype=cdt)
    r_min = 1e-6 if precision == 32 else 1e-11
    with wilson.WilsonContext(dims, precision) as ctx:
        pb, ib = bicgstab_on_gpu(ctx, U, eta, kappa, r_min, 500)
        pc, ic = gu.solve_on_gpu(ctx, U, eta, kappa, r_min, 500)
    po, io = oracle.bicgstab_solve(dims, U.astype(np.complex128), eta.astype(np.complex128), kappa, r_min, 500)
    assert ib["status"] == 0 and ic["status"] == 0 and io["converged"]
    assert abs(ib["iterations"] - io["iterations"]) <= (1 if precision == 32 else 0)
    assert np.linalg.norm(pb - po) / np.linalg.norm(po) < 50 * r_min
    assert np.linalg.norm(pb - pc) / np.linalg.norm(pc) < 50 * r_min


def test_bicgstab_free_field_finite_termination(wilson):
    """pin B-P3 on the GPU (fp64): one plane wave -> exact after 2 iterations; kappa = 0 -> after 1"""
    dims, kappa = (8, 8, 8, 8), 0.12
    U = inputs.gauge_field(0, dims, "unit")
    p = lm.momenta(dims, np.array((1, 2, 0, 3)), -1)
    u = inputs.complex_gaussian(inputs.slice_rng(CFG_TEST + 2, inputs.FIELD_AUX, 0), (4, 3))
    eta = lm.plane_wave(dims, p, u)
    want = lm.plane_wave(dims, p, lm.free_dirac_inverse(p, kappa) @ u)
    with wilson.WilsonContext(dims, 64) as ctx:
        psi, info = bicgstab_on_gpu(ctx, U, eta, kappa, 1e-11, 50)
        assert info["iterations"] == 2 and info["status"] == 0
        assert np.linalg.norm(psi - want) / np.linalg.norm(want) < 1e-10
        src = inputs.source_field(CFG_TEST + 2, dims)
        psi, info = bicgstab_on_gpu(ctx, inputs.gauge_field(CFG_TEST + 2, dims, "haar"), src, 0.0, 1e-12, 10)
        assert info["iterations"] == 1 and np.max(np.abs(psi - src)) < 1e-14


def test_bicgstab_edge_cases(wilson):
    cfg = inputs.CONFIGS[0]
    U, eta = gu.config_fields(0, 32)
    with wilson.WilsonContext(cfg.dims, 32) as ctx:
        psi, info = bicgstab_on_gpu(ctx, U, np.zeros_like(eta), cfg.kappa, 1e-6, 10)
        assert info["status"] == 0 and info["iterations"] == 0 and not psi.any()
        psi, info = bicgstab_on_gpu(ctx, U, eta, cfg.kappa, 1e-6, 0)
        assert info["status"] == 1 and info["iterations"] == 0 and not psi.any()
        psi, info = bicgstab_on_gpu(ctx, U, eta, cfg.kappa, 1e-6, 3)
        assert info["status"] == 1 and info["iterations"] == 3
        a, ia = bicgstab_on_gpu(ctx, U, eta, cfg.kappa, 1e-6, 100)
        ctx.wd_set_poll_interval(1)
        b, ib = bicgstab_on_gpu(ctx, U, eta, cfg.kappa, 1e-6, 100)
        assert a.tobytes() == b.tobytes() and ia["iterations"] == ib["iterations"]   # deterministic, poll-independent


@pytest.mark.parametrize("precision", [32, 64])
def test_bicgstab_32_4_closed_form(wilson, precision):
    """BASELINE volume 32^4 without an oracle solve: pure-gauge links and a Gaussian source; exact solution
    g(x) * free_solve(g^-1 eta) by Fourier transform (pin P8)."""
    dims, kappa = (32, 32, 32, 32), 0.12
    g = inputs.gauge_transform_field(CFG_TEST + 3, dims)
    U = lm.pure_gauge_links(dims, g)
    eta = inputs.source_field(CFG_TEST + 3, dims)
    want = np.einsum("xab,xib->xia", g, lm.free_solve(dims, kappa, np.einsum("xba,xib->xia", np.conj(g), eta), -1))
    cdt = gu.np_complex(precision)
    tol = 1e-6 if precision == 32 else 1e-11
    with wilson.WilsonContext(dims, precision) as ctx:
        psi, info = bicgstab_on_gpu(ctx, U.astype(cdt), eta.astype(cdt), kappa, tol, 2000)
    assert info["status"] == 0
    err = np.linalg.norm(psi - want) / np.linalg.norm(want)
    assert err < (2e-5 if precision == 32 else 1e-9), err
