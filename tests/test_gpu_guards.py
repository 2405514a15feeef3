"""Out-of-bounds checks of our own (-m gpu).  compute-sanitizer is closed on the GPU pool, so every caller-visible
device buffer of a call is carved out of a larger allocation whose guard bands (4 KiB on either side) hold a NaN
pattern with a payload: a kernel that WRITES outside its buffer changes the pattern, one that READS outside it pulls NaNs
into its result.  Lattices are ragged on purpose: volume (and half volume) not a multiple of the 16-site block, extents
not multiples of the tile.  The volume-dependent pad lanes INSIDE the buffers are poisoned too where the call's contract
says they are ignored (inputs of wd_apply / cg_solve / the even-odd calls come from the pack kernels, which zero them)."""
import math

import numpy as np
import pytest

from paper_2111_14958_b200 import inputs
import gpu_util as gu

pytestmark = pytest.mark.gpu

GUARD = 1024          # elements on either side
PATTERN32 = 0x7FC0BEEF
PATTERN64 = 0x7FF80000DEADBEEF
CFG_TEST = 870


@pytest.fixture(scope="module")
def wilson():
    from paper_2111_14958_b200 import build as wbuild
    from paper_2111_14958_b200 import wilson as w

    wbuild.build()
    w.load_library()
    return w


class Guarded:
    """n elements of `dtype` between two guard bands"""

    def __init__(self, like):
        import torch

        self.n = like.numel()
        self.itype = torch.int32 if like.element_size() == 4 else torch.int64
        self.pattern = PATTERN32 if like.element_size() == 4 else PATTERN64
        self.raw = torch.full((self.n + 2 * GUARD,), self.pattern, dtype=self.itype, device="cuda")
        self.t = self.raw[GUARD:GUARD + self.n].view(like.dtype)

    def intact(self):
        lo, hi = self.raw[:GUARD], self.raw[GUARD + self.n:]
        return bool((lo == self.pattern).all()) and bool((hi == self.pattern).all())


def guarded_copy(src):
    g = Guarded(src)
    g.t.copy_(src)
    return g


def all_intact(*gs):
    return all(g.intact() for g in gs)


@pytest.mark.parametrize("precision", [32, 64])
@pytest.mark.parametrize("dims", [(5, 7, 4, 6), (4, 4, 4, 4), (18, 4, 6, 4)])
def test_plain_calls_stay_inside_their_buffers(wilson, dims, precision):
    import torch

    cdt = gu.np_complex(precision)
    r_min = 1e-6 if precision == 32 else 1e-10
    kappa = 0.12
    U = inputs.gauge_field(CFG_TEST, dims, "haar", dtype=cdt)
    eta = inputs.source_field(CFG_TEST, dims, dtype=cdt)
    with wilson.WilsonContext(dims, precision, -1) as ctx:
        Uc, ec = guarded_copy(torch.view_as_real(gu.to_device(U)).reshape(-1)), guarded_copy(torch.view_as_real(gu.to_device(eta)).reshape(-1))
        Un, en, out = Guarded(ctx.empty_gauge()), Guarded(ctx.empty_spinor()), Guarded(ctx.empty_spinor())
        ctx._check(ctx.lib.wd_pack_gauge(ctx._ctx, ctx._p(Uc.t), ctx._p(Un.t)))
        ctx._check(ctx.lib.wd_pack_spinor(ctx._ctx, ctx._p(ec.t), ctx._p(en.t)))
        assert torch.isfinite(Un.t).all() and torch.isfinite(en.t).all()     # pad lanes were written (zeros)
        for tile in range(wilson.load_library().wd_num_tiles()):
            try:
                ctx.wd_set_tile(tile)
            except wilson.WilsonError:
                continue                                                     # not compiled for this precision
            for dag in (0, 1):
                ctx.wd_apply(Un.t, en.t, kappa, dag, out=out.t)
                got = ctx.wd_unpack_spinor(out.t)
                assert torch.isfinite(torch.view_as_real(got)).all(), (tile, dag)
        ctx.wd_set_tile(-1)
        for mode in (1, 2, 6):
            ctx.wd_set_cg_mode(mode)
            _, info = ctx.cg_solve(Un.t, en.t, kappa, r_min, 500, out=out.t)
            assert info["status"] == 0 and torch.isfinite(torch.view_as_real(ctx.wd_unpack_spinor(out.t))).all()
        ctx.wd_set_cg_mode(0)
        _, info = ctx.bicgstab_solve(Un.t, en.t, kappa, r_min, 500, out=out.t)
        assert info["status"] == 0 and torch.isfinite(torch.view_as_real(ctx.wd_unpack_spinor(out.t))).all()
        assert np.isfinite(ctx.wd_norm2(en.t))
        can = Guarded(torch.view_as_real(gu.to_device(eta)).reshape(-1))
        ctx._check(ctx.lib.wd_unpack_spinor(ctx._ctx, ctx._p(out.t), ctx._p(can.t)))
        assert torch.isfinite(can.t).all()
        # the paper's COO arrays
        nnz = ctx.wd_coo_nnz()
        val = Guarded(torch.empty(2 * nnz, dtype=ctx.real_dtype, device="cuda"))
        row = Guarded(torch.empty(nnz, dtype=torch.int32, device="cuda"))
        col = Guarded(torch.empty(nnz, dtype=torch.int32, device="cuda"))
        ctx._check(ctx.lib.wd_coo_assemble(ctx._ctx, ctx._p(Un.t), kappa, 0, ctx._p(val.t), ctx._p(row.t), ctx._p(col.t)))
        assert int(row.t.min()) == 0 and int(row.t.max()) == 12 * ctx.volume - 1
        assert int(col.t.min()) >= 0 and int(col.t.max()) < 12 * ctx.volume
        ctx._check(ctx.lib.wd_coo_spmv(ctx._ctx, nnz, ctx._p(val.t), ctx._p(row.t), ctx._p(col.t), ctx._p(ec.t), ctx._p(can.t)))
        assert torch.isfinite(can.t).all()
        # several right-hand sides: 3 sources in one guarded buffer
        n = en.t.numel()
        em, om = Guarded(torch.empty(3 * n, dtype=ctx.real_dtype, device="cuda")), Guarded(torch.empty(3 * n, dtype=ctx.real_dtype, device="cuda"))
        for j in range(3):
            em.t[j * n:(j + 1) * n] = en.t * (1.0 + j)
        ctx.wd_apply_multi(Un.t, em.t.view(3, n), kappa, False, out=om.t.view(3, n))
        _, infos = ctx.cg_solve_multi(Un.t, em.t.view(3, n), kappa, r_min, 500, out=om.t.view(3, n))
        assert all(i["status"] == 0 for i in infos)
        for j in range(3):
            assert torch.isfinite(torch.view_as_real(ctx.wd_unpack_spinor(om.t[j * n:(j + 1) * n]))).all()
        # 12-real links
        ctx.wd_set_gauge_recon(12)
        U12 = Guarded(ctx.empty_gauge())
        ctx._check(ctx.lib.wd_pack_gauge(ctx._ctx, ctx._p(Uc.t), ctx._p(U12.t)))
        ctx.wd_set_cg_mode(1)
        _, info = ctx.cg_solve(U12.t, en.t, kappa, r_min, 500, out=out.t)
        assert info["status"] == 0 and torch.isfinite(torch.view_as_real(ctx.wd_unpack_spinor(out.t))).all()
        torch.cuda.synchronize()
        assert all_intact(Uc, ec, Un, en, out, can, val, row, col, em, om, U12)
        # inputs were not modified
        assert torch.equal(ec.t, torch.view_as_real(gu.to_device(eta)).reshape(-1))


@pytest.mark.parametrize("precision", [32, 64])
@pytest.mark.parametrize("dims", [(6, 6, 6, 6), (4, 4, 4, 4), (10, 4, 6, 8)])
def test_even_odd_calls_stay_inside_their_buffers(wilson, dims, precision):
    import torch

    cdt = gu.np_complex(precision)
    r_min = 1e-6 if precision == 32 else 1e-10
    kappa = 0.12
    U = inputs.gauge_field(CFG_TEST + 1, dims, "near_identity", dtype=cdt)
    eta = inputs.source_field(CFG_TEST + 1, dims, dtype=cdt)
    with wilson.WilsonContext(dims, precision, -1) as ctx:
        Uc, ec = guarded_copy(torch.view_as_real(gu.to_device(U)).reshape(-1)), guarded_copy(torch.view_as_real(gu.to_device(eta)).reshape(-1))
        Ue, ee, pe, tmp = (Guarded(ctx.empty_eo_gauge()), Guarded(ctx.empty_eo_spinor()), Guarded(ctx.empty_eo_spinor()),
                           Guarded(ctx.empty_eo_spinor()))
        ctx._check(ctx.lib.wd_eo_pack_gauge(ctx._ctx, ctx._p(Uc.t), ctx._p(Ue.t)))
        ctx._check(ctx.lib.wd_eo_pack_spinor(ctx._ctx, ctx._p(ec.t), ctx._p(ee.t)))
        assert torch.isfinite(Ue.t).all() and torch.isfinite(ee.t).all()
        tmp.t.zero_()
        for par in (0, 1):
            for dag in (0, 1):
                ctx.wd_eo_hop(Ue.t, ee.t, tmp.t, par, dag)
        assert torch.isfinite(tmp.t).all()
        _, info = ctx.cg_solve_eo(Ue.t, ee.t, kappa, r_min, 500, out=pe.t)
        assert info["status"] == 0 and torch.isfinite(torch.view_as_real(ctx.wd_eo_unpack_spinor(pe.t))).all()
        for mode in (1, 2):     # seven kernels per iteration, one cooperative launch
            ctx.wd_set_cg_mode(mode)
            _, info = ctx.bicgstab_solve_eo(Ue.t, ee.t, kappa, r_min, 500, out=pe.t)
            assert info["status"] == 0 and info["cg_mode"] == 6 + mode
            assert torch.isfinite(torch.view_as_real(ctx.wd_eo_unpack_spinor(pe.t))).all()
        ctx.wd_set_cg_mode(0)
        can = Guarded(torch.view_as_real(gu.to_device(eta)).reshape(-1))
        ctx._check(ctx.lib.wd_eo_unpack_spinor(ctx._ctx, ctx._p(pe.t), ctx._p(can.t)))
        # the same on 12-real links
        ctx.wd_set_gauge_recon(12)
        U12 = Guarded(ctx.empty_eo_gauge())
        ctx._check(ctx.lib.wd_eo_pack_gauge(ctx._ctx, ctx._p(Uc.t), ctx._p(U12.t)))
        assert torch.isfinite(U12.t).all()
        _, info = ctx.cg_solve_eo(U12.t, ee.t, kappa, r_min, 500, out=pe.t)
        assert info["status"] == 0 and torch.isfinite(torch.view_as_real(ctx.wd_eo_unpack_spinor(pe.t))).all()
        _, info = ctx.bicgstab_solve_eo(U12.t, ee.t, kappa, r_min, 500, out=pe.t)
        assert info["status"] == 0 and torch.isfinite(torch.view_as_real(ctx.wd_eo_unpack_spinor(pe.t))).all()
        torch.cuda.synchronize()
        assert all_intact(Uc, ec, Ue, ee, pe, tmp, can, U12)
        assert torch.equal(ec.t, torch.view_as_real(gu.to_device(eta)).reshape(-1))


# ---------------------------------------------------------------- non-finite inputs, stale pad lanes, max_iter = INT_MAX
@pytest.mark.parametrize("precision", [32, 64])
def test_non_finite_inputs_are_a_breakdown_not_a_convergence(wilson, precision):
    """A NaN link or a NaN / infinite source makes the residual norm NaN; `!(x >= thr)` then ends the loop, and the
    solvers must report WD_BREAKDOWN (status 2, converged 0), never WD_OK with a NaN field (include/wilson_cg.h)."""
    cfg = inputs.CONFIGS[0]
    U, eta = gu.config_fields(0, precision)
    U_bad = U.copy()
    U_bad[17, 2, 1, 1] = np.nan
    eta_nan = eta.copy()
    eta_nan[5, 1, 2] = np.nan
    eta_inf = eta.copy()
    eta_inf[9, 0, 0] = np.inf
    r_min = 1e-6 if precision == 32 else 1e-10
    with wilson.WilsonContext(cfg.dims, precision, cfg.bc_t) as ctx:
        for mode in (1, 2, 6, 9, 10):
            ctx.wd_set_cg_mode(mode)
            for Ux, ex in ((U_bad, eta), (U, eta_nan), (U, eta_inf)):
                _, info = gu.solve_on_gpu(ctx, Ux, ex, cfg.kappa, r_min, 200)
                assert info["status"] == 2 and info["converged"] == 0 and info["iterations"] <= 2, (mode, info)
            # and the ctx is not poisoned: the clean problem still converges
            _, info = gu.solve_on_gpu(ctx, U, eta, cfg.kappa, r_min, 200)
            assert info["status"] == 0 and info["converged"] == 1
        ctx.wd_set_cg_mode(1)
        Un, Ub = ctx.wd_pack_gauge(gu.to_device(U)), ctx.wd_pack_gauge(gu.to_device(U_bad))
        en, eb = ctx.wd_pack_spinor(gu.to_device(eta)), ctx.wd_pack_spinor(gu.to_device(eta_nan))
        for Ux, ex in ((Ub, en), (Un, eb)):
            _, info = ctx.bicgstab_solve(Ux, ex, cfg.kappa, r_min, 200)
            assert info["status"] == 2 and info["converged"] == 0, info
        for mode in (1, 2):     # seven / five kernels per iteration, and the one-launch even-odd BiCGSTAB
            ctx.wd_set_cg_mode(mode)
            for Ux, ex in ((U_bad, eta), (U, eta_nan)):
                Ue = ctx.wd_eo_pack_gauge(gu.to_device(Ux))
                ee = ctx.wd_eo_pack_spinor(gu.to_device(ex))
                _, info = ctx.bicgstab_solve_eo(Ue, ee, cfg.kappa, r_min, 200)
                assert info["status"] == 2 and info["converged"] == 0, (mode, info)
                if mode == 1:
                    _, info = ctx.cg_solve_eo(Ue, ee, cfg.kappa, r_min, 200)
                    assert info["status"] == 2 and info["converged"] == 0, info


@pytest.mark.parametrize("precision", [32, 64])
@pytest.mark.parametrize("dims", [(14, 14, 14, 14), (6, 6, 6, 10)])
def test_even_odd_solvers_ignore_stale_pad_lanes(wilson, oracle, dims, precision):
    """V/2 is not a multiple of the 16-site block here.  The even-odd solvers run on half-length views of the ctx work
    vectors; a full-lattice solve that stopped after one iteration leaves O(1) data where those views have their pad
    lanes.  It must not leak into the recurrence: iteration counts and residuals equal the oracle's as on a fresh ctx."""
    assert (int(np.prod(dims)) // 2) % 16 != 0
    cdt = gu.np_complex(precision)
    kappa, r_min = 0.12, (1e-6 if precision == 32 else 1e-10)
    U = inputs.gauge_field(777, dims, "haar", dtype=cdt)
    eta = inputs.source_field(777, dims, dtype=cdt)
    U64, eta64 = U.astype(np.complex128), eta.astype(np.complex128)
    _, ioc = oracle.cg_solve_eo(dims, U64, eta64, kappa, r_min, 500, -1)
    _, iob = oracle.bicgstab_solve_eo(dims, U64, eta64, kappa, r_min, 500, -1)
    with wilson.WilsonContext(dims, precision, -1) as ctx:
        ctx.wd_set_cg_mode(1)                       # kernel-per-phase drivers (the one-launch kernels own their vectors)
        Un = ctx.wd_pack_gauge(gu.to_device(U))
        en = ctx.wd_pack_spinor(gu.to_device(eta))
        # poison: every work vector holds O(1) data at all lanes the stencil and the vector kernels ever wrote
        ctx.cg_solve(Un, en, kappa, r_min, 1)
        ctx.bicgstab_solve(Un, en, kappa, r_min, 1)
        Ue = ctx.wd_eo_pack_gauge(gu.to_device(U))
        ee = ctx.wd_eo_pack_spinor(gu.to_device(eta))
        pb, ib = ctx.bicgstab_solve_eo(Ue, ee, kappa, r_min, 500)
        psi_b = gu.to_host(ctx.wd_eo_unpack_spinor(pb))
        pc, ic = ctx.cg_solve_eo(Ue, ee, kappa, r_min, 500)
        psi_c = gu.to_host(ctx.wd_eo_unpack_spinor(pc))
    slack = 0 if precision == 64 else max(1, int(0.05 * iob["iterations"] + 0.5))
    assert ib["status"] == 0 and abs(ib["iterations"] - iob["iterations"]) <= slack, (ib, iob)
    assert ic["status"] == 0 and abs(ic["iterations"] - ioc["iterations"]) <= math.floor(0.02 * ioc["iterations"] + 0.5)
    for name, psi in (("bicgstab_eo", psi_b), ("cg_eo", psi_c)):
        res = oracle.true_residual(dims, U64, eta64, psi.astype(np.complex128), kappa, -1)
        assert res < 2.0 * r_min, (name, res)


@pytest.mark.parametrize("precision", [32, 64])
def test_bicgstab_ignores_the_pad_lanes_of_its_source(wilson, oracle, precision):
    """5 x 7 x 4 x 6 = 840 sites = 52.5 blocks.  The source is the output of wd_apply into a buffer full of NaN: its
    real sites hold D eta, its 8 pad lanes stay NaN (the stencil never writes them).  rhat = that source enters two dot
    products per iteration: they must skip the pad lanes."""
    import torch

    dims, kappa = (5, 7, 4, 6), 0.12
    cdt = gu.np_complex(precision)
    r_min = 1e-6 if precision == 32 else 1e-10
    U = inputs.gauge_field(778, dims, "haar", dtype=cdt)
    eta = inputs.source_field(778, dims, dtype=cdt)
    with wilson.WilsonContext(dims, precision, 1) as ctx:
        ctx.wd_set_cg_mode(1)
        Un = ctx.wd_pack_gauge(gu.to_device(U))
        en = ctx.wd_pack_spinor(gu.to_device(eta))
        src = torch.full_like(en, float("nan"))
        ctx.wd_apply(Un, en, kappa, False, out=src)
        assert bool(torch.isnan(src).any())                      # the pad lanes
        src_can = gu.to_host(ctx.wd_unpack_spinor(src))
        assert np.isfinite(src_can).all()
        for solve in (ctx.bicgstab_solve, ctx.cg_solve):
            psi_n, info = solve(Un, src, kappa, r_min, 500)
            psi = gu.to_host(ctx.wd_unpack_spinor(psi_n))
            assert info["status"] == 0 and np.isfinite(psi).all(), info
            # D psi = D eta  =>  psi = eta
            assert np.linalg.norm(psi - eta) / np.linalg.norm(eta) < 4.0 * r_min * (1 + 8 * kappa) / (1 - 8 * kappa)
    U64, s64 = U.astype(np.complex128), src_can.astype(np.complex128)
    _, io = oracle.bicgstab_solve(dims, U64, s64, kappa, r_min, 500, 1)
    assert abs(info["iterations"] - oracle.cg_solve(dims, U64, s64, kappa, r_min, 500, 1)[1]["iterations"]) <= 1
    assert io["converged"]


def test_max_iter_int_max_means_no_limit(wilson):
    """max_iter = INT_MAX: max_iter + 1 must not overflow, the history stays bounded, the solve converges as usual"""
    cfg = inputs.CONFIGS[0]
    U, eta = gu.config_fields(0, 32)
    with wilson.WilsonContext(cfg.dims, 32, cfg.bc_t) as ctx:
        ref = None
        for mode in (1, 2, 6, 9, 10):
            ctx.wd_set_cg_mode(mode)
            psi, info = gu.solve_on_gpu(ctx, U, eta, cfg.kappa, cfg.r_min, 2 ** 31 - 1)
            assert info["status"] == 0 and info["converged"] == 1 and 20 < info["iterations"] < 40
            ref = ref or info["iterations"]
            assert info["iterations"] == ref
        Un = ctx.wd_pack_gauge(gu.to_device(U))
        en = ctx.wd_pack_spinor(gu.to_device(eta))
        _, ib = ctx.bicgstab_solve(Un, en, cfg.kappa, cfg.r_min, 2 ** 31 - 1)
        assert ib["status"] == 0


def test_contexts_on_their_own_streams_run_concurrently(wilson):
    """include/wilson_cg.h: "use one ctx per host thread / stream".  Two host threads, each with its own context on its own
    stream, solve at the same time (ctypes releases the GIL during a call): every driver of cg_solve and BiCGSTAB, each
    with the per-context scratch of its reductions and the process-wide occupancy tables.  Every result must be
    bit-identical to the same solve run alone (the reductions are deterministic)."""
    import threading

    import torch

    jobs = [(0, 32, 1), (1, 32, 2), (0, 64, 6), (0, 32, 9), (2, 32, 10), (1, 32, 1), (2, 32, 0), (1, 64, 0)]
    prepared = []
    for ci, precision, mode in jobs:
        cfg = inputs.CONFIGS[ci]
        U, eta = gu.config_fields(ci, precision)
        r_min = cfg.r_min if precision == 32 else 1e-10
        stream = torch.cuda.Stream()
        with torch.cuda.stream(stream):
            ctx = wilson.WilsonContext(cfg.dims, precision, cfg.bc_t, stream=stream)
            ctx.wd_set_cg_mode(mode)
            Un = ctx.wd_pack_gauge(gu.to_device(U))
            en = ctx.wd_pack_spinor(gu.to_device(eta))
            out, outb = ctx.empty_spinor(), ctx.empty_spinor()
            _, info = ctx.cg_solve(Un, en, cfg.kappa, r_min, cfg.max_iter, out=out)
            _, infob = ctx.bicgstab_solve(Un, en, cfg.kappa, r_min, cfg.max_iter, out=outb)
            stream.synchronize()
            prepared.append((ctx, stream, cfg, r_min, Un, en, out.clone(), info, outb.clone(), infob))
    torch.cuda.synchronize()
    errors = []

    def worker(items, rounds):
        try:
            for _ in range(rounds):
                for ctx, stream, cfg, r_min, Un, en, want, info, wantb, infob in items:
                    with torch.cuda.stream(stream):
                        got, gi = ctx.cg_solve(Un, en, cfg.kappa, r_min, cfg.max_iter)
                        gotb, gib = ctx.bicgstab_solve(Un, en, cfg.kappa, r_min, cfg.max_iter)
                        stream.synchronize()
                        if gi["iterations"] != info["iterations"] or gi["cg_mode"] != info["cg_mode"] or not torch.equal(got, want):
                            errors.append(("cg", cfg.index, ctx.precision, gi, info))
                        if gib["iterations"] != infob["iterations"] or not torch.equal(gotb, wantb):
                            errors.append(("bicgstab", cfg.index, ctx.precision, gib, infob))
        except Exception as e:  # noqa: BLE001 - reported by the main thread
            errors.append(("exception", repr(e)))

    threads = [threading.Thread(target=worker, args=(prepared[k::2], 6)) for k in range(2)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    for p in prepared:
        p[0].close()
    assert not errors, errors[:3]


@pytest.mark.parametrize("precision", [32, 64])
def test_host_buffer_calls_stay_inside_their_host_buffers(wilson, oracle, precision):
    """cg_solve_host, wd_apply_host and the split-phase calls move their fields in slabs of whole 16-site blocks; on a lattice
    whose volume is not a multiple of 16 (and smaller than 8 slabs of blocks would like) the last slab must stop at V: the host
    buffers sit between guard bands that must not change (output) and whose NaNs must not be read (inputs)."""
    dims, kappa, bc_t = (5, 7, 4, 6), 0.12, -1
    V = int(np.prod(dims))
    cdt = gu.np_complex(precision)
    r_min = 1e-6 if precision == 32 else 1e-10
    U = inputs.gauge_field(CFG_TEST + 30, dims, "haar", dtype=cdt)
    eta = inputs.source_field(CFG_TEST + 30, dims, dtype=cdt)
    g = 64

    def guarded(a):
        big = np.full((a.shape[0] + 2 * g,) + a.shape[1:], np.nan + 1j * np.nan, dtype=a.dtype)
        big[g:g + a.shape[0]] = a
        return big, big[g:g + a.shape[0]]

    Ub, Uv = guarded(U)
    eb, ev = guarded(eta)
    ob, ov = guarded(np.zeros_like(eta))
    ob[:g] = 7.0
    ob[g + V:] = 7.0
    with wilson.WilsonContext(dims, precision, bc_t) as ctx:
        psi_d, info_d = gu.solve_on_gpu(ctx, U, eta, kappa, r_min, 500)
        _, info_h = ctx.cg_solve_host(Uv, ev, kappa, r_min, 500, out=ov)
        assert info_h["iterations"] == info_d["iterations"] and ov.tobytes() == psi_d.tobytes()
        assert (ob[:g] == 7.0).all() and (ob[g + V:] == 7.0).all()
        ov[:] = 0
        out_d = gu.apply_on_gpu(ctx, U, eta, kappa, True)
        ctx.wd_apply_host(Uv, ev, kappa, True, out=ov)
        assert ov.tobytes() == out_d.tobytes() and (ob[:g] == 7.0).all() and (ob[g + V:] == 7.0).all()
        ov[:] = 0
        ctx.cg_solve_host_begin(Uv, ev)
        info_s = ctx.cg_solve_host_run(kappa, r_min, 500, ov)
        ctx.cg_solve_host_wait()
        assert info_s["iterations"] == info_d["iterations"] and ov.tobytes() == psi_d.tobytes()
        assert (ob[:g] == 7.0).all() and (ob[g + V:] == 7.0).all()
    assert np.isnan(Ub[:g]).all() and np.isnan(eb[g + V:]).all()        # the inputs were not written either
