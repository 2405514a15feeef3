"""-m gpu parity tests: the CUDA path, called through the C ABI (ctypes binding), against the fp64
CPU oracle on the same seeded inputs.

Tolerances (BASELINE.json north_star; readings G15, G16, G18 in DESIGN.md):
  * wd_apply: max over sites of |out_gpu(x) - out_ref(x)|_2 / |out_ref(x)|_2  <= 1e-5 (fp32), 1e-12 (fp64);
  * cg_solve: iteration count within +-2 % of the oracle's, final TRUE residual |eta - D psi|/|eta|
    (evaluated by the oracle's fp64 D) within a factor 2 of the oracle's;
  * pack / unpack are permutations: bit-exact.
For fp32 runs the oracle consumes the fp32-rounded inputs promoted to fp64, so both sides see the
identical operator and source.
"""
import ctypes
import json
import math
import os

import numpy as np
import pytest

from paper_2111_14958_b200 import inputs
import gpu_util as gu
import lattice_math as lm

pytestmark = pytest.mark.gpu

TOL_APPLY = {32: 1e-5, 64: 1e-12}
GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
CFG_TEST = 700


@pytest.fixture(scope="module")
def wilson():
    import torch

    assert torch.cuda.is_available(), "the -m gpu tests need a CUDA device"
    from paper_2111_14958_b200 import build as wbuild
    from paper_2111_14958_b200 import wilson as w

    wbuild.build()
    w.load_library()
    return w


def iters_close(a, b):
    return abs(a - b) <= max(0.02 * b, 0.0) + 1e-9 or abs(a - b) <= math.floor(0.02 * b + 0.5)


# ---------------------------------------------------------------- a0: layouts
@pytest.mark.parametrize("precision", [32, 64])
@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (6, 4, 10, 8), (5, 7, 4, 6), (14, 14, 14, 14)])
def test_pack_unpack_are_exact_permutations(wilson, precision, dims):
    V = int(np.prod(dims))
    cdt = gu.np_complex(precision)
    rdt = np.float32 if precision == 32 else np.float64
    psi = inputs.source_field(CFG_TEST, dims, dtype=cdt, field=inputs.FIELD_AUX)
    U = inputs.gauge_field(CFG_TEST, dims, "haar", dtype=cdt)
    with wilson.WilsonContext(dims, precision) as ctx:
        pn = ctx.wd_pack_spinor(gu.to_device(psi))
        Un = ctx.wd_pack_gauge(gu.to_device(U))
        back = gu.to_host(ctx.wd_unpack_spinor(pn))
        pn_h, Un_h = gu.to_host(pn), gu.to_host(Un)
    assert back.tobytes() == psi.tobytes()
    # native layout (include/wilson_cg.h): blocks of 16 lexicographic sites; inside a block the spinor is NSP
    # planes of 128-bit vectors, the gauge field 36 planes (mu*9 + a*3+b) of one complex; pad lanes are zero
    nblk = (V + 15) // 16
    Vp = nblk * 16
    nsp, w = (6, 4) if precision == 32 else (12, 2)
    want = np.zeros((Vp, nsp, w), dtype=rdt)
    want[:V] = psi.view(rdt).reshape(V, nsp, w)
    want = want.reshape(nblk, 16, nsp, w).transpose(0, 2, 1, 3)
    assert pn_h.size == Vp * 24 and pn_h.tobytes() == np.ascontiguousarray(want).tobytes()
    # gauge block = 4 links x (9 complex x 16 sites); fp64: 9 planes of one complex; fp32: 4 planes of float4
    # (reals 4q..4q+3) followed by one plane of float2 (reals 16, 17)
    u18 = np.zeros((Vp, 4, 18), dtype=rdt)
    u18[:V] = U.view(rdt).reshape(V, 4, 18)
    u18 = u18.reshape(nblk, 16, 4, 18).transpose(0, 2, 1, 3)          # [blk][mu][site][18]
    if precision == 64:
        want_u = u18.reshape(nblk, 4, 16, 9, 2).transpose(0, 1, 3, 2, 4)
    else:
        head = u18[..., :16].reshape(nblk, 4, 16, 4, 4).transpose(0, 1, 3, 2, 4).reshape(nblk, 4, 256)
        tail = u18[..., 16:].reshape(nblk, 4, 32)
        want_u = np.concatenate([head, tail], axis=2)
    assert Un_h.size == Vp * 72 and Un_h.tobytes() == np.ascontiguousarray(want_u).tobytes()


# ---------------------------------------------------------------- a7: wd_apply
def _apply_case(wilson, oracle, dims, links, kappa, precision, bc_t, cfg_seed, tile=None):
    cdt = gu.np_complex(precision)
    U = inputs.gauge_field(cfg_seed, dims, links, dtype=cdt)
    psi = inputs.source_field(cfg_seed, dims, dtype=cdt, field=inputs.FIELD_AUX)
    worst = 0.0
    with wilson.WilsonContext(dims, precision, bc_t) as ctx:
        if tile is not None:
            ctx.wd_set_tile(tile)
        for dagger in (False, True):
            got = gu.apply_on_gpu(ctx, U, psi, kappa, dagger)
            want = oracle.wd_apply(dims, U.astype(np.complex128), psi.astype(np.complex128), kappa, dagger, bc_t)
            site, glob = lm.per_site_rel_err(got, want)
            assert site <= TOL_APPLY[precision], (dims, precision, dagger, bc_t, tile, site, glob)
            worst = max(worst, site)
    return worst


@pytest.mark.parametrize("precision", [32, 64])
@pytest.mark.parametrize("cfg_index", [0, 1, 2])
def test_wd_apply_baseline_configs(wilson, oracle, cfg_index, precision):
    cfg = inputs.CONFIGS[cfg_index]
    _apply_case(wilson, oracle, cfg.dims, cfg.links, cfg.kappa, precision, cfg.bc_t, cfg.index)


@pytest.mark.parametrize("precision", [32, 64])
@pytest.mark.parametrize("bc_t", [-1, 1])
@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (6, 4, 10, 8), (5, 7, 4, 6), (18, 4, 6, 4), (4, 4, 4, 34)])
def test_wd_apply_ragged_and_anisotropic(wilson, oracle, dims, bc_t, precision):
    """extents that are not multiples of any tile edge, all four extents different, both boundary conditions"""
    _apply_case(wilson, oracle, dims, "haar", 0.12, precision, bc_t, CFG_TEST + 1)


@pytest.mark.parametrize("precision", [32, 64])
def test_every_tile_shape(wilson, oracle, precision):
    n = len(wilson.tile_shapes())
    ran = 0
    for tile in range(n):
        for dims in [(14, 14, 14, 14), (16, 8, 8, 4)]:
            try:
                _apply_case(wilson, oracle, dims, "haar", 0.12, precision, -1, CFG_TEST + 2, tile=tile)
                ran += 1
            except wilson.WilsonError as e:
                assert e.code == -1 and not wilson.tile_infos()[tile][5 if precision == 32 else 6]  # row not compiled for this precision
    assert ran >= 8


def test_wd_apply_free_field_plane_wave(wilson):
    """closed form, no oracle: D on a plane wave in the free field (pin P3) at a volume spanning many tiles"""
    dims, kappa = (16, 12, 8, 20), 0.124
    U = inputs.gauge_field(0, dims, "unit")
    n = np.array([3, 5, 1, 7])
    p = lm.momenta(dims, n, -1)
    u = inputs.complex_gaussian(inputs.slice_rng(CFG_TEST, inputs.FIELD_AUX, 0), (4, 3))
    psi = lm.plane_wave(dims, p, u)
    want = np.einsum("ij,xja->xia", lm.free_dirac_symbol(p, kappa), psi)
    want_dag = np.einsum("ij,xja->xia", lm.free_dirac_symbol(p, kappa).conj().T, psi)
    with wilson.WilsonContext(dims, 64) as ctx:
        assert lm.per_site_rel_err(gu.apply_on_gpu(ctx, U, psi, kappa, False), want)[0] < 1e-12
        assert lm.per_site_rel_err(gu.apply_on_gpu(ctx, U, psi, kappa, True), want_dag)[0] < 1e-12


@pytest.mark.parametrize("precision", [32, 64])
def test_wd_apply_32_4_sampled_sites(wilson, oracle, precision):
    """BASELINE config 3 at full size, bench launch configuration; the oracle evaluates sampled sites one by one"""
    cfg = inputs.CONFIGS[3]
    U, psi = gu.config_fields(3, precision)
    V = cfg.volume
    rng = np.random.Generator(np.random.PCG64(5))
    lx, ly, lz, lt = cfg.dims
    edge = [0, lx - 1, lx, V - 1, V - lx, lx * ly * lz * (lt - 1), lx * ly * lz - 1, lx * ly - 1]
    sites = np.unique(np.concatenate([edge, rng.choice(V, 4000, replace=False)])).astype(np.int64)
    U64, psi64 = U.astype(np.complex128), psi.astype(np.complex128)
    with wilson.WilsonContext(cfg.dims, precision, cfg.bc_t) as ctx:
        for dagger in (False, True):
            got = gu.apply_on_gpu(ctx, U, psi, cfg.kappa, dagger)[sites]
            want = oracle.wd_apply_sites(cfg.dims, U64, psi64, cfg.kappa, sites, dagger, cfg.bc_t)
            assert lm.per_site_rel_err(got, want)[0] <= TOL_APPLY[precision]


def test_wd_apply_config4_sampled_sites(wilson, oracle):
    """BASELINE config 4 (48^3 x 96, fp32: the paper's quoted production volume, and the workload bench.py
    times) in the launch configuration of the bench: D and D-dagger at > 20 000 sampled sites plus the lattice corners,
    both t-boundary slices (where the antiperiodic sign acts), the last 16-site block and the first and last site of
    every tile row of the first tile column, one by one against the oracle; per-site relative error <= 1e-5
    (BASELINE.json north_star)."""
    cfg = inputs.CONFIGS[4]
    U, psi = gu.config_fields(4, 32)
    V = cfg.volume
    lx, ly, lz, lt = cfg.dims
    rng = np.random.Generator(np.random.PCG64(11))
    corners = [x + lx * (y + ly * (z + lz * t)) for x in (0, lx - 1) for y in (0, ly - 1) for z in (0, lz - 1)
               for t in (0, lt - 1)]
    slab = lx * ly * lz
    t_first = rng.choice(slab, 1500, replace=False)                       # t = 0: backward t hop wraps
    t_last = slab * (lt - 1) + rng.choice(slab, 1500, replace=False)      # t = Lt-1: forward t hop wraps
    last_block = np.arange(V - 16, V)
    tile_rows = np.array([x + lx * (y + ly * (z + lz * t)) for x in (0, 15, 16, lx - 1) for y in (0, 1, 2, ly - 1)
                          for z in (0, 1, 2, lz - 1) for t in (0, 1, 2, lt - 1)])
    sites = np.unique(np.concatenate([corners, t_first, t_last, last_block, tile_rows,
                                      rng.choice(V, 20000, replace=False)])).astype(np.int64)
    assert sites.size > 20000
    U64, psi64 = U.astype(np.complex128), psi.astype(np.complex128)
    with wilson.WilsonContext(cfg.dims, 32, cfg.bc_t) as ctx:
        Un = ctx.wd_pack_gauge(gu.to_device(U))
        pn = ctx.wd_pack_spinor(gu.to_device(psi))
        dev_sites = gu.to_device(sites)
        for dagger in (False, True):
            got = gu.to_host(ctx.wd_unpack_spinor(ctx.wd_apply(Un, pn, cfg.kappa, dagger))[dev_sites])
            want = oracle.wd_apply_sites(cfg.dims, U64, psi64, cfg.kappa, sites, dagger, cfg.bc_t)
            site_err, glob_err = lm.per_site_rel_err(got, want)
            assert site_err <= TOL_APPLY[32], (dagger, site_err, glob_err)


def test_largest_supported_volume(wilson, oracle):
    """96^2 x 64 x 96 = 56.6 M sites: 36 V = 2.04e9 is just below the 2^31 limit of the 32-bit plane indexing that
    wd_create enforces (16 GB of links, 5.4 GB per spinor in fp32).  wd_apply D and D-dagger at sampled sites, among them
    the last sites of the lattice (largest indices) and its corners, one by one against the oracle; then the whole
    cg_solve, its true residual evaluated by the oracle's fp64 D on the full lattice."""
    dims, kappa, r_min = (96, 96, 64, 96), 0.124, 1e-6
    V = int(np.prod(dims))
    assert 0.94 * 2 ** 31 < 36 * V < 2 ** 31
    U = inputs.gauge_field(CFG_TEST + 9, dims, "near_identity", dtype=np.complex64)
    eta = inputs.source_field(CFG_TEST + 9, dims, dtype=np.complex64)
    U64, eta64 = U.astype(np.complex128), eta.astype(np.complex128)
    rng = np.random.Generator(np.random.PCG64(7))
    lx, ly, lz, lt = dims
    edge = [0, lx - 1, lx, V - 1, V - 2, V - lx, lx * ly * lz * (lt - 1), lx * ly * lz - 1, lx * ly - 1, V // 2, V - 17]
    sites = np.unique(np.concatenate([edge, rng.choice(V, 3000, replace=False)])).astype(np.int64)
    with wilson.WilsonContext(dims, 32, -1) as ctx:
        Un = ctx.wd_pack_gauge(gu.to_device(U))
        en = ctx.wd_pack_spinor(gu.to_device(eta))
        for dagger in (False, True):
            got = gu.to_host(ctx.wd_unpack_spinor(ctx.wd_apply(Un, en, kappa, dagger))[gu.to_device(sites)])
            want = oracle.wd_apply_sites(dims, U64, eta64, kappa, sites, dagger, -1)
            assert lm.per_site_rel_err(got, want)[0] <= TOL_APPLY[32]
        psi_n, info = ctx.cg_solve(Un, en, kappa, r_min, 5000)
        psi = gu.to_host(ctx.wd_unpack_spinor(psi_n))
        del Un, en, psi_n
    assert info["status"] == 0 and info["cg_mode"] == 1 and 50 < info["iterations"] < 400
    res = oracle.true_residual(dims, U64, eta64, psi.astype(np.complex128), kappa, -1)
    assert res < 2.0 * r_min, res
    assert abs(info["eta_norm2"] / (24.0 * V) - 1.0) < 1e-3        # pin P9 at this size


# ---------------------------------------------------------------- the shared-memory link pipeline (wilson_tma.cuh)
@pytest.mark.parametrize("precision", [32, 64])
@pytest.mark.parametrize("dims,bc_t", [((16, 4, 4, 4), -1), ((32, 8, 4, 8), 1), ((48, 4, 8, 6), -1), ((16, 12, 8, 10), -1)])
def test_link_staging_is_bit_identical_and_matches_oracle(wilson, oracle, dims, bc_t, precision):
    """wd_set_link_staging(row): the gauge field reaches the stencil through bulk copies into a shared-memory ring, both
    uses of every link served from there.  Same arithmetic in the same order: wd_apply D and D-dagger are bit-identical to
    the kernel that reads the links through L1 for every compiled row that covers the lattice (several tiles per CTA, so the
    ring wraps across tile boundaries; both boundary conditions; x extent of one, two and three 16-site blocks), and
    within the wd_apply tolerance of the oracle.  A row that does not cover the lattice is refused."""
    cdt = gu.np_complex(precision)
    U = inputs.gauge_field(CFG_TEST + 11, dims, "haar", dtype=cdt)
    psi = inputs.source_field(CFG_TEST + 11, dims, dtype=cdt, field=inputs.FIELD_AUX)
    U64, psi64 = U.astype(np.complex128), psi.astype(np.complex128)
    ran = 0
    with wilson.WilsonContext(dims, precision, bc_t) as ctx:
        Un = ctx.wd_pack_gauge(gu.to_device(U))
        pn = ctx.wd_pack_spinor(gu.to_device(psi))
        ctx.wd_set_link_staging(-1)      # the reference: links through L1
        ref = {dag: gu.to_host(ctx.wd_unpack_spinor(ctx.wd_apply(Un, pn, 0.12, dag))) for dag in (False, True)}
        for dag in (False, True):
            want = oracle.wd_apply(dims, U64, psi64, 0.12, dag, bc_t)
            assert lm.per_site_rel_err(ref[dag], want)[0] <= TOL_APPLY[precision]
        for row, info in enumerate(wilson.staging_rows()):
            covers = info[7 if precision == 32 else 8] and all(dims[d] % info[d] == 0 for d in range(4))
            if not covers:
                with pytest.raises(wilson.WilsonError):
                    ctx.wd_set_link_staging(row)
                continue
            ctx.wd_set_link_staging(row)
            assert ctx.wd_get_link_staging() == row
            for dag in (False, True):
                for _ in range(2):      # twice: the barriers are re-initialised by every launch
                    got = gu.to_host(ctx.wd_unpack_spinor(ctx.wd_apply(Un, pn, 0.12, dag)))
                    assert got.tobytes() == ref[dag].tobytes(), (row, info, dag)
            ran += 1
            ctx.wd_set_link_staging(-1)
            assert ctx.wd_get_link_staging() == -1
    assert ran >= 1


@pytest.mark.parametrize("precision", [32, 64])
def test_cg_solve_with_link_staging(wilson, oracle, precision):
    """the three-kernel CG with every stencil pass (a2, a3, a6) on the staged kernel: iteration count, residual history and
    true residual against the oracle (config 1, 8^4 is too narrow: a 16 x 8 x 8 x 8 lattice with config 1's recipe), and
    against the unstaged solve (per-site arithmetic identical, only the grouping of the reduction partials differs)."""
    dims, kappa, bc_t = (16, 8, 8, 8), 0.124, -1
    r_min = 1e-6 if precision == 32 else 1e-10
    cdt = gu.np_complex(precision)
    U = inputs.gauge_field(CFG_TEST + 12, dims, "near_identity", dtype=cdt)
    eta = inputs.source_field(CFG_TEST + 12, dims, dtype=cdt)
    U64, eta64 = U.astype(np.complex128), eta.astype(np.complex128)
    psi_o, info_o = oracle.cg_solve(dims, U64, eta64, kappa, r_min, 1000, bc_t, history=True)
    res_o = oracle.true_residual(dims, U64, eta64, psi_o, kappa, bc_t)
    ran = 0
    with wilson.WilsonContext(dims, precision, bc_t) as ctx:
        ctx.wd_set_cg_mode(1)
        ctx.wd_set_link_staging(-1)
        psi0, info0 = gu.solve_on_gpu(ctx, U, eta, kappa, r_min, 1000)
        for row, info in list(enumerate(wilson.staging_rows())) + [(-2, None)]:
            if row == -2:          # the automatic choice (the default of a fresh ctx)
                ctx.wd_set_link_staging(-2)
                assert ctx.wd_get_link_staging() == (-1 if precision == 32 else 2)
                psi, inf = gu.solve_on_gpu(ctx, U, eta, kappa, r_min, 1000)
                assert inf["status"] == 0 and inf["iterations"] == info0["iterations"]
                assert np.linalg.norm(psi - psi0) <= (1e-5 if precision == 32 else 1e-12) * np.linalg.norm(psi0)
                continue
            if not (info[7 if precision == 32 else 8] and all(dims[d] % info[d] == 0 for d in range(4))):
                continue
            ctx.wd_set_link_staging(row)
            psi, inf = gu.solve_on_gpu(ctx, U, eta, kappa, r_min, 1000)
            hist = ctx.wd_cg_history()
            assert inf["status"] == 0 and inf["cg_mode"] == 1
            assert iters_close(inf["iterations"], info_o["iterations"]) and inf["iterations"] == info0["iterations"]
            res = oracle.true_residual(dims, U64, eta64, psi.astype(np.complex128), kappa, bc_t)
            assert res <= 2.0 * res_o, (row, res, res_o)
            n = min(len(hist), len(info_o["rr_history"])) // 2
            rel = np.abs(hist[:n] - info_o["rr_history"][:n]) / info_o["rr_history"][:n]
            assert np.max(rel) < (2e-2 if precision == 32 else 1e-6)
            assert np.linalg.norm(psi - psi0) <= (1e-5 if precision == 32 else 1e-12) * np.linalg.norm(psi0)
            ran += 1
    assert ran >= 1


# ---------------------------------------------------------------- reductions
@pytest.mark.parametrize("precision", [32, 64])
def test_norm2_matches_oracle_and_is_deterministic(wilson, oracle, precision):
    dims = (14, 14, 14, 14)
    a = inputs.source_field(CFG_TEST + 3, dims, dtype=gu.np_complex(precision))
    with wilson.WilsonContext(dims, precision) as ctx:
        an = ctx.wd_pack_spinor(gu.to_device(a))
        got = [ctx.wd_norm2(an) for _ in range(3)]
    want = oracle.norm2(a.astype(np.complex128))
    assert got[0] == got[1] == got[2]
    assert abs(got[0] - want) <= (1e-6 if precision == 32 else 1e-13) * want
    assert abs(want / (2 * 12 * np.prod(dims)) - 1) < 0.01  # pin P9: re, im each N(0,1)


# ---------------------------------------------------------------- a1-a6: cg_solve
def _cg_case(wilson, oracle, cfg, precision, r_min, poll=None, mode=0):
    """mode: 0 automatic, 1 three kernels per iteration, 2 whole solve in one cooperative launch (thread per site), 6 one
    cooperative launch with the hopping sum of a site split over four warps"""
    U, eta = gu.config_fields(cfg.index, precision)
    U64, eta64 = U.astype(np.complex128), eta.astype(np.complex128)
    with wilson.WilsonContext(cfg.dims, precision, cfg.bc_t) as ctx:
        if poll:
            ctx.wd_set_poll_interval(poll)
        ctx.wd_set_cg_mode(mode)
        psi, info = gu.solve_on_gpu(ctx, U, eta, cfg.kappa, r_min, cfg.max_iter)
        hist = ctx.wd_cg_history()
    if mode:
        assert info["cg_mode"] == mode
        # one-launch drivers: the solve kernel + the one-warp kernel that writes the scalars to the pinned host mirror
        assert info["kernel_launches"] == 2 if mode in (2, 6, 9, 10) else info["kernel_launches"] >= 3 * info["iterations"] + 2
    psi_o, info_o = oracle.cg_solve(cfg.dims, U64, eta64, cfg.kappa, r_min, cfg.max_iter, cfg.bc_t, history=True)
    res_gpu = oracle.true_residual(cfg.dims, U64, eta64, psi.astype(np.complex128), cfg.kappa, cfg.bc_t)
    res_orc = oracle.true_residual(cfg.dims, U64, eta64, psi_o, cfg.kappa, cfg.bc_t)
    assert info["status"] == 0 and info["converged"] == 1 and info_o["converged"]
    assert iters_close(info["iterations"], info_o["iterations"]), (info["iterations"], info_o["iterations"])
    assert res_gpu <= 2.0 * res_orc, (res_gpu, res_orc)
    assert res_gpu < 2.0 * r_min
    # the device-side record of the recursed residual follows the oracle's history
    n = min(len(hist), len(info_o["rr_history"]))
    assert len(hist) == info["iterations"] + 1
    rel = np.abs(hist[:n] - info_o["rr_history"][:n]) / info_o["rr_history"][:n]
    assert rel[0] < (1e-6 if precision == 32 else 1e-13)
    assert np.max(rel[: max(2, n // 2)]) < (2e-2 if precision == 32 else 1e-6)
    # solutions agree to what the tolerance allows: |dpsi| <= |D^-1| (|r_gpu| + |r_orc|)
    diff = np.linalg.norm(psi - psi_o) / np.linalg.norm(psi_o)
    assert diff < 4.0 * r_min / (1.0 - 8.0 * cfg.kappa) * (1 + 8 * cfg.kappa)
    return info, info_o, res_gpu, res_orc


def _resident_covers(cfg, precision):
    """mode 9 (lattice resident in the shared memory of a cluster): V / nc a power of two <= 256 (fp32) / 128 (fp64), nc <= 16"""
    return cfg.index == 0 or (cfg.index == 1 and precision == 32)


@pytest.mark.parametrize("mode", [1, 2, 6, 9, 10])
@pytest.mark.parametrize("cfg_index", [0, 1, 2])
def test_cg_solve_fp32_baseline_configs(wilson, oracle, cfg_index, mode):
    """the CG drivers: three kernels per iteration (mode 1), the two one-launch cooperative kernels (modes 2, 6) and the
    shared-memory-resident cluster kernel (mode 9: 4^4 on one CTA, 8^4 on a 16-CTA cluster)"""
    cfg = inputs.CONFIGS[cfg_index]
    if mode == 9 and not _resident_covers(cfg, 32):
        with wilson.WilsonContext(cfg.dims, 32, cfg.bc_t) as ctx, pytest.raises(wilson.WilsonError):
            ctx.wd_set_cg_mode(9)
        return
    _cg_case(wilson, oracle, cfg, 32, cfg.r_min, mode=mode)


@pytest.mark.parametrize("mode", [1, 2, 6, 9, 10])
@pytest.mark.parametrize("cfg_index", [0, 1, 2])
def test_cg_solve_fp64_tight(wilson, oracle, cfg_index, mode):
    cfg = inputs.CONFIGS[cfg_index]
    if (mode == 9 and not _resident_covers(cfg, 64)) or (mode == 10 and cfg_index == 2):
        # (mode 10 in fp64: 14^4 has 686 tiles of 16x2x2x1, more than the 592 CTAs that can be co-resident)
        with wilson.WilsonContext(cfg.dims, 64, cfg.bc_t) as ctx, pytest.raises(wilson.WilsonError):
            ctx.wd_set_cg_mode(mode)
        return
    _cg_case(wilson, oracle, cfg, 64, 1e-10, mode=mode)


@pytest.mark.parametrize("precision", [32, 64])
@pytest.mark.parametrize("dims,bc_t", [((4, 4, 4, 8), 1), ((8, 4, 4, 4), -1), ((4, 8, 4, 8), -1), ((8, 8, 4, 4), 1), ((4, 4, 8, 16), -1)])
def test_cg_resident_cluster_sizes(wilson, oracle, dims, bc_t, precision):
    """mode 9 on anisotropic lattices: clusters of 2, 4, 8 and 16 CTAs (fp32: 512 ... 2048 sites at 256 per CTA; fp64: 128 per
    CTA), slabs that cut the z and t directions at different places, both boundary conditions; against the oracle and
    repeatable bit for bit"""
    V = int(np.prod(dims))
    if V // (256 if precision == 32 else 128) > 16:
        with wilson.WilsonContext(dims, precision, bc_t) as ctx, pytest.raises(wilson.WilsonError):
            ctx.wd_set_cg_mode(9)
        return
    cdt = gu.np_complex(precision)
    tol = 1e-6 if precision == 32 else 1e-10
    U = inputs.gauge_field(CFG_TEST + 31, dims, "haar", dtype=cdt)
    eta = inputs.source_field(CFG_TEST + 31, dims, dtype=cdt)
    U64, eta64 = U.astype(np.complex128), eta.astype(np.complex128)
    psi_o, info_o = oracle.cg_solve(dims, U64, eta64, 0.12, tol, 500, bc_t)
    outs = []
    with wilson.WilsonContext(dims, precision, bc_t) as ctx:
        ctx.wd_set_cg_mode(9)
        for _ in range(2):
            psi, info = gu.solve_on_gpu(ctx, U, eta, 0.12, tol, 500)
            outs.append(psi.tobytes())
        assert info["status"] == 0 and info["cg_mode"] == 9 and info["kernel_launches"] == 2
    assert outs[0] == outs[1]
    assert iters_close(info["iterations"], info_o["iterations"])
    res = oracle.true_residual(dims, U64, eta64, psi.astype(np.complex128), 0.12, bc_t)
    assert res <= 2.0 * oracle.true_residual(dims, U64, eta64, psi_o, 0.12, bc_t)


def test_cg_automatic_mode_by_volume(wilson):
    """4^4 and 8^4 (fp32) take the shared-memory-resident kernel (one CTA, a cluster of sixteen with exported half-spinors; 4^4
    fp64: a cluster of two), the rest of the paper's range a one-launch cooperative kernel (gauge field in shared
    memory: mode 10; fp64 8^4, which fits no cluster: the split kernel), 32^4 the three-kernel loop"""
    for ci, precision, want in ((0, 32, 9), (1, 32, 9), (2, 32, 10), (0, 64, 9), (1, 64, 6)):
        cfg = inputs.CONFIGS[ci]
        U, eta = gu.config_fields(ci, precision)
        with wilson.WilsonContext(cfg.dims, precision, cfg.bc_t) as ctx:
            _, info = gu.solve_on_gpu(ctx, U, eta, cfg.kappa, cfg.r_min, cfg.max_iter)
        assert info["cg_mode"] == want and info["kernel_launches"] == 2
    # in between: the resident kernel wherever V / nc is a power of two that fits a CTA (fp32 <= 4096 sites, fp64 <= 2048)
    for dims, precision, want in (((8, 4, 4, 8), 32, 9), ((4, 8, 8, 8), 32, 9), ((4, 4, 8, 8), 64, 9), ((4, 8, 8, 8), 64, 9),
                                  ((6, 6, 6, 6), 32, 10), ((8, 8, 8, 16), 32, 10),
                                  ((16, 16, 4, 4), 32, 10)):   # 16 CTAs, but 1024 exports per CTA do not fit beside the slabs
        cdt = gu.np_complex(precision)
        U = inputs.gauge_field(CFG_TEST + 7, dims, "haar", dtype=cdt)
        eta = inputs.source_field(CFG_TEST + 7, dims, dtype=cdt)
        with wilson.WilsonContext(dims, precision) as ctx:
            _, info = gu.solve_on_gpu(ctx, U, eta, 0.12, 1e-6, 500)
        assert info["status"] == 0 and info["cg_mode"] == want, (dims, precision, info["cg_mode"])


@pytest.mark.parametrize("precision", [32, 64])
def test_cg_onelaunch_ragged_lattice(wilson, oracle, precision):
    """both one-launch kernels on extents that no tile divides, periodic t as well"""
    for dims, bc_t in (((6, 4, 10, 8), -1), ((5, 7, 4, 6), 1), ((18, 4, 6, 4), -1)):
        cdt = gu.np_complex(precision)
        U = inputs.gauge_field(CFG_TEST + 6, dims, "near_identity", dtype=cdt)
        eta = inputs.source_field(CFG_TEST + 6, dims, dtype=cdt)
        tol = 1e-6 if precision == 32 else 1e-11
        U64, eta64 = U.astype(np.complex128), eta.astype(np.complex128)
        psi_o, info_o = oracle.cg_solve(dims, U64, eta64, 0.12, tol, 500, bc_t)
        for mode in (2, 6, 10):
            with wilson.WilsonContext(dims, precision, bc_t) as ctx:
                ctx.wd_set_cg_mode(mode)
                psi, info = gu.solve_on_gpu(ctx, U, eta, 0.12, tol, 500)
            assert info["status"] == 0 and info["cg_mode"] == mode and iters_close(info["iterations"], info_o["iterations"])
            res = oracle.true_residual(dims, U64, eta64, psi.astype(np.complex128), 0.12, bc_t)
            assert res <= 2.0 * oracle.true_residual(dims, U64, eta64, psi_o, 0.12, bc_t)


def _random_lattices(n, seed):
    """n seeded lattices with extents in [4, 19], skewed towards small ones (the oracle has to finish in seconds)"""
    rng = np.random.Generator(np.random.PCG64(seed))
    out = []
    while len(out) < n:
        dims = tuple(int(d) for d in rng.choice([4, 5, 6, 7, 8, 9, 10, 11, 12, 13, 14, 16, 17, 19], size=4))
        if 256 <= int(np.prod(dims)) <= 20000:
            out.append((dims, int(rng.choice([-1, 1]))))
    return out


@pytest.mark.parametrize("precision", [32, 64])
def test_random_lattices_operator_and_every_cg_driver(wilson, oracle, precision):
    """16 seeded lattices with unrelated, mostly odd extents, either boundary condition: D and D-dagger per site against the
    oracle, then cg_solve with the automatic choice and with every driver that accepts the lattice (a driver may refuse a
    lattice it has no launch configuration for, with WD_ERR_ARG; it must not accept it and be wrong)."""
    tol = 1e-6 if precision == 32 else 1e-11
    drivers_run = {m: 0 for m in (0, 1, 2, 6, 9, 10)}
    for k, (dims, bc_t) in enumerate(_random_lattices(16, 20211114)):
        cdt = gu.np_complex(precision)
        links = "haar" if k % 2 else "near_identity"
        U = inputs.gauge_field(CFG_TEST + 20, dims, links, dtype=cdt)
        eta = inputs.source_field(CFG_TEST + 20, dims, dtype=cdt)
        U64, eta64 = U.astype(np.complex128), eta.astype(np.complex128)
        kappa = 0.11 if links == "haar" else 0.122
        with wilson.WilsonContext(dims, precision, bc_t) as ctx:
            for dagger in (False, True):
                got = gu.apply_on_gpu(ctx, U, eta, kappa, dagger)
                want = oracle.wd_apply(dims, U64, eta64, kappa, dagger, bc_t)
                assert lm.per_site_rel_err(got, want)[0] <= TOL_APPLY[precision], (dims, bc_t, dagger)
        psi_o, info_o = oracle.cg_solve(dims, U64, eta64, kappa, tol, 400, bc_t)
        res_o = oracle.true_residual(dims, U64, eta64, psi_o, kappa, bc_t)
        assert info_o["converged"]
        for mode in drivers_run:
            with wilson.WilsonContext(dims, precision, bc_t) as ctx:
                try:
                    ctx.wd_set_cg_mode(mode)
                    psi, info = gu.solve_on_gpu(ctx, U, eta, kappa, tol, 400)
                except wilson.WilsonError as e:
                    assert e.code == -1 and mode in (9, 10), (dims, mode, str(e))
                    continue
            drivers_run[mode] += 1
            assert info["status"] == 0 and info["converged"] == 1, (dims, mode, info)
            assert iters_close(info["iterations"], info_o["iterations"]), (dims, mode, info["iterations"], info_o["iterations"])
            res = oracle.true_residual(dims, U64, eta64, psi.astype(np.complex128), kappa, bc_t)
            assert res <= 2.0 * res_o, (dims, mode, res, res_o)
    assert all(drivers_run[m] == 16 for m in (0, 1, 2, 6)) and drivers_run[10] >= 8, drivers_run


def test_cg_result_independent_of_poll_interval_and_repeatable(wilson):
    cfg = inputs.CONFIGS[1]
    U, eta = gu.config_fields(1, 32)
    outs = []
    for poll in (1, 7, 32, 7):
        with wilson.WilsonContext(cfg.dims, 32, cfg.bc_t) as ctx:
            ctx.wd_set_cg_mode(1)
            ctx.wd_set_poll_interval(poll)
            psi, info = gu.solve_on_gpu(ctx, U, eta, cfg.kappa, cfg.r_min, cfg.max_iter)
            outs.append((psi.tobytes(), info["iterations"], info["rel_residual"]))
    assert all(o == outs[0] for o in outs)
    # the one-launch kernel is repeatable too (fixed-order sums of the per-CTA partials in every CTA)
    outs = []
    for _ in range(3):
        with wilson.WilsonContext(cfg.dims, 32, cfg.bc_t) as ctx:
            ctx.wd_set_cg_mode(2)
            psi, info = gu.solve_on_gpu(ctx, U, eta, cfg.kappa, cfg.r_min, cfg.max_iter)
            outs.append((psi.tobytes(), info["iterations"], info["rel_residual"]))
    assert all(o == outs[0] for o in outs)
    for mode9 in (9, 10):
        outs = []
        for _ in range(3):
            with wilson.WilsonContext(cfg.dims, 32, cfg.bc_t) as ctx:
                ctx.wd_set_cg_mode(mode9)     # 8^4: a 16-CTA cluster, partial sums through distributed shared memory
                psi, info = gu.solve_on_gpu(ctx, U, eta, cfg.kappa, cfg.r_min, cfg.max_iter)
                outs.append((psi.tobytes(), info["iterations"], info["rel_residual"]))
        assert all(o == outs[0] for o in outs)
    outs = []
    for _ in range(3):
        with wilson.WilsonContext(cfg.dims, 32, cfg.bc_t) as ctx:
            ctx.wd_set_cg_mode(6)
            psi, info = gu.solve_on_gpu(ctx, U, eta, cfg.kappa, cfg.r_min, cfg.max_iter)
            outs.append((psi.tobytes(), info["iterations"], info["rel_residual"]))
    assert all(o == outs[0] for o in outs)


def test_wd_apply_repeat_is_wd_apply(wilson):
    """the measurement aid enqueues the same launches as wd_apply: same output, a positive device time, argument checks"""
    cfg = inputs.CONFIGS[2]
    U, eta = gu.config_fields(2, 32)
    with wilson.WilsonContext(cfg.dims, 32, cfg.bc_t) as ctx:
        Un = ctx.wd_pack_gauge(gu.to_device(U))
        en = ctx.wd_pack_spinor(gu.to_device(eta))
        for dag in (False, True):
            want = gu.to_host(ctx.wd_unpack_spinor(ctx.wd_apply(Un, en, cfg.kappa, dag)))
            out = ctx.empty_spinor()
            ms = ctx.wd_apply_repeat(Un, en, cfg.kappa, dag, reps=20, out=out)
            assert 0.0 < ms < 1.0
            assert np.array_equal(gu.to_host(ctx.wd_unpack_spinor(out)), want)
        with pytest.raises(wilson.WilsonError):
            ctx.wd_apply_repeat(Un, en, cfg.kappa, False, reps=0)
        with pytest.raises(wilson.WilsonError):
            ctx.wd_apply_repeat(Un, en, cfg.kappa, False, reps=3, out=en)


@pytest.mark.parametrize("mode", [1, 2, 6, 9, 10])
def test_cg_edge_cases(wilson, oracle, mode):
    cfg = inputs.CONFIGS[0]
    U, eta = gu.config_fields(0, 64)
    with wilson.WilsonContext(cfg.dims, 64, cfg.bc_t) as ctx:
        ctx.wd_set_cg_mode(mode)
        # eta = 0: psi = 0, no iterations, OK
        psi, info = gu.solve_on_gpu(ctx, U, np.zeros_like(eta), cfg.kappa, 1e-8, 100)
        assert info["status"] == 0 and info["iterations"] == 0 and not psi.any()
        # max_iter = 0: nothing iterated, psi = D-dagger 0 = 0, not converged
        psi, info = gu.solve_on_gpu(ctx, U, eta, cfg.kappa, 1e-8, 0)
        assert info["status"] == 1 and info["iterations"] == 0 and not psi.any()
        # max_iter reached: exactly the oracle's iterate after 5 loop bodies
        psi, info = gu.solve_on_gpu(ctx, U, eta, cfg.kappa, 1e-12, 5)
        psi_o, info_o = oracle.cg_solve(cfg.dims, U, eta, cfg.kappa, 1e-12, 5, cfg.bc_t)
        assert info["status"] == 1 and info["converged"] == 0 and info["iterations"] == 5 == info_o["iterations"]
        assert np.linalg.norm(psi - psi_o) / np.linalg.norm(psi_o) < 1e-12
        assert abs(info["rel_residual"] - info_o["rel_residual"]) < 1e-12 * info_o["rel_residual"] + 1e-15
        # kappa = 0: D = 1, one iteration, psi = eta (pin P7)
        psi, info = gu.solve_on_gpu(ctx, U, eta, 0.0, 1e-12, 10)
        assert info["iterations"] == 1 and np.max(np.abs(psi - eta)) < 1e-14
        # r_min >= 1: the loop condition fails at once
        psi, info = gu.solve_on_gpu(ctx, U, eta, cfg.kappa, 1.5, 10)
        assert info["status"] == 0 and info["iterations"] == 0


@pytest.mark.parametrize("dims,precision", [((8, 8, 8, 8), 32), ((4, 8, 8, 8), 64), ((4, 8, 8, 8), 32)])
def test_cg_edge_cases_on_clusters_with_exported_half_spinors(wilson, oracle, dims, precision):
    """the degenerate cases on the resident kernel of 8 / 16 CTAs (cg_resident_ex_kernel; automatic for these lattices): the
    paths that leave the loop at once still have to export y for the final D-dagger and keep every CTA in the barriers"""
    cdt = gu.np_complex(precision)
    tol = 1e-6 if precision == 32 else 1e-12
    U = inputs.gauge_field(CFG_TEST + 11, dims, "haar", dtype=cdt)
    eta = inputs.source_field(CFG_TEST + 11, dims, dtype=cdt)
    U64, eta64 = U.astype(np.complex128), eta.astype(np.complex128)
    for bc_t in (-1, 1):
        with wilson.WilsonContext(dims, precision, bc_t) as ctx:
            psi, info = gu.solve_on_gpu(ctx, U, np.zeros_like(eta), 0.12, 1e-8, 100)
            assert info["cg_mode"] == 9 and info["status"] == 0 and info["iterations"] == 0 and not psi.any()
            psi, info = gu.solve_on_gpu(ctx, U, eta, 0.12, 1e-8, 0)
            assert info["status"] == 1 and info["iterations"] == 0 and not psi.any()
            psi, info = gu.solve_on_gpu(ctx, U, eta, 0.12, 1e-12, 5)
            psi_o, info_o = oracle.cg_solve(dims, U64, eta64, 0.12, 1e-12, 5, bc_t)
            assert info["status"] == 1 and info["converged"] == 0 and info["iterations"] == 5 == info_o["iterations"]
            assert np.linalg.norm(psi - psi_o) / np.linalg.norm(psi_o) < (2e-6 if precision == 32 else 1e-12)
            psi, info = gu.solve_on_gpu(ctx, U, eta, 0.0, tol, 10)
            assert info["iterations"] == 1 and np.max(np.abs(psi - eta)) < (1e-6 if precision == 32 else 1e-14)
            psi, info = gu.solve_on_gpu(ctx, U, eta, 0.12, 1.5, 10)
            assert info["status"] == 0 and info["iterations"] == 0
            # a NaN in the source is a breakdown, not a convergence
            bad = eta.copy()
            bad[17, 2, 1] = np.nan
            _, info = gu.solve_on_gpu(ctx, U, bad, 0.12, 1e-6, 50)
            assert info["status"] == 2 and info["converged"] == 0
            # the whole solve against the oracle, and repeatable bit for bit
            psi, info = gu.solve_on_gpu(ctx, U, eta, 0.12, tol if precision == 32 else 1e-10, 500)
            psi2, info2 = gu.solve_on_gpu(ctx, U, eta, 0.12, tol if precision == 32 else 1e-10, 500)
            psi_o, info_o = oracle.cg_solve(dims, U64, eta64, 0.12, tol if precision == 32 else 1e-10, 500, bc_t)
            assert info["status"] == 0 and iters_close(info["iterations"], info_o["iterations"]) and psi.tobytes() == psi2.tobytes()
            res = oracle.true_residual(dims, U64, eta64, psi.astype(np.complex128), 0.12, bc_t)
            assert res <= 2.0 * oracle.true_residual(dims, U64, eta64, psi_o, 0.12, bc_t)


def test_cg_free_field_finite_termination(wilson):
    """pin P8: K plane waves with distinct |D(p)|^2 terminate after exactly K iterations, exact solution known"""
    dims, kappa = (8, 8, 8, 8), 0.12
    U = inputs.gauge_field(0, dims, "unit")
    rng = inputs.slice_rng(CFG_TEST + 4, inputs.FIELD_AUX, 0)
    eta = np.zeros((int(np.prod(dims)), 4, 3), dtype=np.complex128)
    want = np.zeros_like(eta)
    modes = [(0, 0, 0, 0), (1, 2, 0, 3), (3, 1, 2, 1)]
    for n in modes:
        p = lm.momenta(dims, np.array(n), -1)
        u = inputs.complex_gaussian(rng, (4, 3))
        eta += lm.plane_wave(dims, p, u)
        want += lm.plane_wave(dims, p, lm.free_dirac_inverse(p, kappa) @ u)
    with wilson.WilsonContext(dims, 64) as ctx:
        psi, info = gu.solve_on_gpu(ctx, U, eta, kappa, 1e-11, 50)
    assert info["iterations"] == len(modes)
    assert np.linalg.norm(psi - want) / np.linalg.norm(want) < 1e-10


@pytest.mark.parametrize("precision", [32, 64])
def test_cg_point_source_closed_form_32_4(wilson, precision):
    """T3 / pin P8 at BASELINE volume 32^4, no oracle CG needed: pure-gauge links U = g(x) g(x+mu)^dagger
    (every link non-trivial) and a point source; the exact solution is g(x) times the free propagator (FFT)."""
    dims, kappa = (32, 32, 32, 32), 0.12
    V = int(np.prod(dims))
    g = inputs.gauge_transform_field(CFG_TEST + 5, dims)
    U = lm.pure_gauge_links(dims, g)
    x0 = (3, 31, 0, 17)
    s0 = int(lm.site_index(dims, np.array(x0)))
    u = inputs.complex_gaussian(inputs.slice_rng(CFG_TEST + 5, inputs.FIELD_AUX, 0), (4, 3))
    eta = np.zeros((V, 4, 3), dtype=np.complex128)
    eta[s0] = u
    # D[U] psi = eta  <=>  D_free (g^-1 psi) = g^-1 eta
    free = lm.free_point_propagator(dims, kappa, x0, np.einsum("ba,ib->ia", np.conj(g[s0]), u), -1)
    want = np.einsum("xab,xib->xia", g, free)
    cdt = gu.np_complex(precision)
    tol = 1e-6 if precision == 32 else 1e-11
    with wilson.WilsonContext(dims, precision) as ctx:
        psi, info = gu.solve_on_gpu(ctx, U.astype(cdt), eta.astype(cdt), kappa, tol, 2000)
    assert info["status"] == 0
    err = np.linalg.norm(psi - want) / np.linalg.norm(want)
    assert err < (2e-5 if precision == 32 else 1e-9), err


def _golden(name):
    path = os.path.join(GOLDEN, name)
    if not os.path.exists(path):
        pytest.skip(f"{name} not generated yet (tests/golden/make_golden.py)")
    with open(path) as f:
        return json.load(f)


@pytest.mark.parametrize("cfg_index,precision", [(3, 32), (3, 64), (4, 32)])
def test_cg_large_configs_against_stored_oracle(wilson, oracle, cfg_index, precision):
    """BASELINE configs 3 and 4 at full size.  The oracle's CG takes minutes to an hour there, so its result
    is stored by tests/golden/make_golden.py (oracle only); the true residual of the GPU solution is still
    evaluated live by the oracle's fp64 D on the full lattice."""
    gold = _golden(f"cg_config{cfg_index}_fp{precision}.json")
    cfg = inputs.CONFIGS[cfg_index]
    U, eta = gu.config_fields(cfg_index, precision)
    with wilson.WilsonContext(cfg.dims, precision, cfg.bc_t) as ctx:
        psi, info = gu.solve_on_gpu(ctx, U, eta, cfg.kappa, gold["r_min"], cfg.max_iter)
        hist = ctx.wd_cg_history()
    assert info["status"] == 0
    assert iters_close(info["iterations"], gold["iterations"]), (info["iterations"], gold["iterations"])
    assert abs(info["eta_norm2"] - gold["eta_norm2"]) < (1e-6 if precision == 32 else 1e-12) * gold["eta_norm2"]
    res = oracle.true_residual(cfg.dims, U.astype(np.complex128), eta.astype(np.complex128),
                               psi.astype(np.complex128), cfg.kappa, cfg.bc_t)
    assert res <= 2.0 * gold["true_residual"], (res, gold["true_residual"])
    sites = np.array(gold["sample_sites"])
    want = (np.array(gold["psi_samples_re"]) + 1j * np.array(gold["psi_samples_im"])).reshape(-1, 4, 3)
    diff = np.linalg.norm(psi[sites] - want) / np.linalg.norm(want)
    assert diff < 4.0 * gold["r_min"] / (1.0 - 8.0 * cfg.kappa) * (1 + 8 * cfg.kappa), diff
    n = min(len(hist), len(gold["rr_history"])) // 2
    gh = np.array(gold["rr_history"][:n])
    assert np.max(np.abs(hist[:n] - gh) / gh) < (5e-2 if precision == 32 else 1e-5)


# ---------------------------------------------------------------- host-buffer forms and errors
@pytest.mark.parametrize("precision", [32, 64])
def test_host_forms_equal_device_forms(wilson, precision):
    cfg = inputs.CONFIGS[1]
    U, eta = gu.config_fields(1, precision)
    with wilson.WilsonContext(cfg.dims, precision, cfg.bc_t) as ctx:
        psi_d, info_d = gu.solve_on_gpu(ctx, U, eta, cfg.kappa, cfg.r_min, cfg.max_iter)
        psi_h, info_h = ctx.cg_solve_host(U, eta, cfg.kappa, cfg.r_min, cfg.max_iter)
        assert psi_h.tobytes() == psi_d.tobytes() and info_h["iterations"] == info_d["iterations"]
        assert info_h["total_ms"] >= info_h["gpu_ms"] > 0 and info_h["kernel_launches"] >= 4
        out_d = gu.apply_on_gpu(ctx, U, eta, cfg.kappa, True)
        out_h = ctx.wd_apply_host(None, eta, cfg.kappa, True)  # reuses the cached gauge field
        assert out_h.tobytes() == out_d.tobytes()


@pytest.mark.parametrize("precision,ci", [(32, 1), (32, 2), (64, 1)])
def test_split_phase_host_solves_pipelined_over_two_contexts(wilson, oracle, precision, ci):
    """cg_solve_host_begin / _run / _wait (include/wilson_cg.h): a queue of DIFFERENT systems (own gauge field and source
    each) pipelined over two contexts on two streams, one host thread.  Every solution must be bit-identical to
    cg_solve_host on the same inputs, and the first one is checked against the oracle like every other solve."""
    import torch

    cfg = inputs.CONFIGS[ci]
    n = 5
    cdt = gu.np_complex(precision)
    r_min = cfg.r_min if precision == 32 else 1e-10
    systems = []
    for k in range(n):
        U = inputs.gauge_field(CFG_TEST + 40 + k, cfg.dims, cfg.links, cfg.eps, dtype=cdt)
        eta = inputs.source_field(CFG_TEST + 50 + k, cfg.dims, dtype=cdt)
        systems.append((torch.from_numpy(U).pin_memory(), torch.from_numpy(eta).pin_memory()))
    V = int(np.prod(cfg.dims))
    outs = [torch.zeros((V, 4, 3), dtype=torch.complex64 if precision == 32 else torch.complex128).pin_memory() for _ in range(n)]
    with wilson.WilsonContext(cfg.dims, precision, cfg.bc_t) as ref_ctx:
        want = [ref_ctx.cg_solve_host(U, eta, cfg.kappa, r_min, cfg.max_iter) for U, eta in systems]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    ctxs = [wilson.WilsonContext(cfg.dims, precision, cfg.bc_t, stream=s) for s in streams]
    try:
        infos = []
        ctxs[0].cg_solve_host_begin(*systems[0])
        with pytest.raises(wilson.WilsonError):
            ctxs[0].cg_solve_host_begin(*systems[0])              # already staged
        with pytest.raises(wilson.WilsonError):
            ctxs[1].cg_solve_host_run(cfg.kappa, r_min, cfg.max_iter, outs[1])   # nothing staged on this ctx
        ctxs[1].cg_solve_host_wait()                               # nothing pending: a no-op
        for i in range(n):
            if i + 1 < n:
                ctxs[(i + 1) % 2].cg_solve_host_begin(*systems[i + 1])
            infos.append(ctxs[i % 2].cg_solve_host_run(cfg.kappa, r_min, cfg.max_iter, outs[i]))
            if i > 0:
                ctxs[(i - 1) % 2].cg_solve_host_wait()
        ctxs[(n - 1) % 2].cg_solve_host_wait()
        # the binding's helper does the same choreography
        outs2 = [torch.zeros_like(o).pin_memory() for o in outs]
        infos2 = wilson.cg_solve_host_queue(ctxs, systems, cfg.kappa, r_min, cfg.max_iter, outs2)
        assert [d["iterations"] for d in infos2] == [d["iterations"] for d in infos]
        assert all(torch.equal(a, b) for a, b in zip(outs, outs2))
        for i in range(n):
            psi_w, info_w = want[i]
            assert infos[i]["status"] == 0 and infos[i]["iterations"] == info_w["iterations"]
            assert outs[i].numpy().tobytes() == np.asarray(psi_w).tobytes(), i
        # queues of length 0 and 1, and an output buffer reused two solves later
        assert wilson.cg_solve_host_queue(ctxs, [], cfg.kappa, r_min, cfg.max_iter, []) == []
        one = wilson.cg_solve_host_queue(ctxs, systems[:1], cfg.kappa, r_min, cfg.max_iter, [outs2[0]])
        assert one[0]["iterations"] == want[0][1]["iterations"] and torch.equal(outs2[0], outs[0])
        ring = [outs2[0], outs2[1]]
        infos3 = wilson.cg_solve_host_queue(ctxs, systems[:4], cfg.kappa, r_min, cfg.max_iter, [ring[i % 2] for i in range(4)])
        assert [d["iterations"] for d in infos3] == [d["iterations"] for d in infos[:4]]
        assert torch.equal(ring[0], outs[2]) and torch.equal(ring[1], outs[3])      # the last writers of the two buffers
        # the gauge field of the previous call on a ctx is reused when U_host is None
        ctxs[1].cg_solve_host_begin(None, systems[3][1])           # ctx 1 last held U of system 3 (the ring run above)
        info = ctxs[1].cg_solve_host_run(cfg.kappa, r_min, cfg.max_iter, outs2[4])
        ctxs[1].cg_solve_host_wait()
        assert info["iterations"] == want[3][1]["iterations"]
        assert outs2[4].numpy().tobytes() == np.asarray(want[3][0]).tobytes()
    finally:
        for c in ctxs:
            c.close()
    U0, eta0 = systems[0][0].numpy(), systems[0][1].numpy()
    U64, eta64 = U0.astype(np.complex128), eta0.astype(np.complex128)
    psi_o, info_o = oracle.cg_solve(cfg.dims, U64, eta64, cfg.kappa, r_min, cfg.max_iter, cfg.bc_t)
    assert iters_close(want[0][1]["iterations"], info_o["iterations"])
    res = oracle.true_residual(cfg.dims, U64, eta64, np.asarray(want[0][0]).astype(np.complex128), cfg.kappa, cfg.bc_t)
    res_o = oracle.true_residual(cfg.dims, U64, eta64, psi_o, cfg.kappa, cfg.bc_t)
    assert res <= 2.0 * res_o


def test_error_codes(wilson):
    cfg = inputs.CONFIGS[0]
    U, eta = gu.config_fields(0, 32)
    with wilson.WilsonContext(cfg.dims, 32) as ctx:
        Un = ctx.wd_pack_gauge(gu.to_device(U))
        en = ctx.wd_pack_spinor(gu.to_device(eta))
        with pytest.raises(wilson.WilsonError) as e:
            ctx.wd_apply(Un, en, cfg.kappa, False, out=en)  # out aliases psi
        assert e.value.code == -1
        with pytest.raises(wilson.WilsonError):
            ctx.wd_apply(Un, en, float("nan"), False)
        with pytest.raises(wilson.WilsonError):
            ctx.cg_solve(Un, en, cfg.kappa, 0.0, 10)
        with pytest.raises(wilson.WilsonError):
            ctx.cg_solve(Un, en, cfg.kappa, 1e-6, -1)
        with pytest.raises(wilson.WilsonError):
            ctx.wd_set_tile(99)
        assert ctx.lib.wd_apply(ctx._ctx, None, None, None, 0.1, 0) == -1
        assert b"wd_apply" in ctx.lib.wd_last_error(ctx._ctx)
        # the ctx is still usable after errors
        assert ctx.wd_norm2(en) > 0
    with pytest.raises(wilson.WilsonError) as e:
        wilson.WilsonContext((4, 4, 3, 4))
    assert e.value.code == -2
