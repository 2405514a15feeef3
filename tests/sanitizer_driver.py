"""Small driver for compute-sanitizer (tier T4): every entry point of the C ABI once, on lattices
small enough for memcheck / racecheck / initcheck / synccheck, including ragged ones (volume and half volume not
multiples of the 16-site block, extents not multiples of the tile):

    PYTORCH_NO_CUDA_MEMORY_CACHING=1 compute-sanitizer --tool memcheck python tests/sanitizer_driver.py [--big]

(without the caching allocator every tensor is its own cudaMalloc, so an out-of-bounds access cannot hide inside a pool).
compute-sanitizer is closed on the GPU pool this repo was built on; there the driver runs plainly (it is also a
whole-API smoke run with the caching allocator off) and tests/test_gpu_guards.py looks for out-of-bounds accesses with
guard bands instead.  Results are only checked for finiteness and convergence here; parity is the job of the -m gpu tests."""
import os
import sys

import numpy as np
import torch

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
from paper_2111_14958_b200 import inputs, wilson  # noqa: E402

SEED = 900


def fields(dims, links, cdt):
    return inputs.gauge_field(SEED, dims, links, dtype=cdt), inputs.source_field(SEED, dims, dtype=cdt)


def plain(dims, links, precision, kappa=0.12):
    cdt = np.complex64 if precision == 32 else np.complex128
    r_min = 1e-6 if precision == 32 else 1e-10
    U, eta = fields(dims, links, cdt)
    with wilson.WilsonContext(dims, precision, -1) as ctx:
        Un = ctx.wd_pack_gauge(torch.from_numpy(U).cuda())
        en = ctx.wd_pack_spinor(torch.from_numpy(eta).cuda())
        back = ctx.wd_unpack_spinor(en).cpu().numpy()
        assert np.array_equal(back, eta)
        for dag in (0, 1):
            out = ctx.wd_apply(Un, en, kappa, dag)
            assert torch.isfinite(out).all()
        assert ctx.wd_norm2(en) > 0
        for mode in (1, 2, 6):
            ctx.wd_set_cg_mode(mode)
            _, info = ctx.cg_solve(Un, en, kappa, r_min, 500)
            assert info["status"] == 0, info
        ctx.wd_set_cg_mode(0)
        ctx.wd_set_sweep(1)
        _, info = ctx.cg_solve(Un, en, kappa, r_min, 500)
        assert info["status"] == 0
        ctx.wd_set_sweep(0)
        ctx.wd_cg_history()
        _, info = ctx.bicgstab_solve(Un, en, kappa, r_min, 500)
        assert info["status"] == 0, info
        # several right-hand sides
        em = torch.stack([en * (1.0 + 0.5 * j) for j in range(3)]).contiguous()
        om = ctx.wd_apply_multi(Un, em, kappa, False)
        assert torch.isfinite(om).all()
        _, infos = ctx.cg_solve_multi(Un, em, kappa, r_min, 500)
        assert all(i["status"] == 0 for i in infos)
        # the paper's COO route
        val, row, col = ctx.wd_coo_assemble(Un, kappa, False)
        got = ctx.wd_coo_spmv(val, row, col, torch.from_numpy(eta).cuda())
        assert torch.isfinite(torch.view_as_real(got)).all()
        # host-buffer forms
        psi_h, info = ctx.cg_solve_host(U, eta, kappa, r_min, 500)
        assert info["status"] == 0 and np.isfinite(psi_h).all()
        out_h = ctx.wd_apply_host(None, eta, kappa, False)
        assert np.isfinite(out_h).all()
        # 12-real links
        ctx.wd_set_gauge_recon(12)
        U12 = ctx.wd_pack_gauge(torch.from_numpy(U).cuda())
        out = ctx.wd_apply(U12, en, kappa, 0)
        assert torch.isfinite(out).all()
        ctx.wd_set_cg_mode(1)
        _, info = ctx.cg_solve(U12, en, kappa, r_min, 500)
        assert info["status"] == 0
    print("plain", dims, links, precision, "ok", flush=True)


def even_odd(dims, links, precision, kappa=0.12):
    cdt = np.complex64 if precision == 32 else np.complex128
    r_min = 1e-6 if precision == 32 else 1e-10
    U, eta = fields(dims, links, cdt)
    with wilson.WilsonContext(dims, precision, -1) as ctx:
        Ue = ctx.wd_eo_pack_gauge(torch.from_numpy(U).cuda())
        ee = ctx.wd_eo_pack_spinor(torch.from_numpy(eta).cuda())
        assert np.array_equal(ctx.wd_eo_unpack_spinor(ee).cpu().numpy(), eta)
        tmp = torch.zeros_like(ee)
        for par in (0, 1):
            for dag in (0, 1):
                ctx.wd_eo_hop(Ue, ee, tmp, par, dag)
        assert torch.isfinite(tmp).all()
        _, info = ctx.cg_solve_eo(Ue, ee, kappa, r_min, 500)
        assert info["status"] == 0, info
        _, info = ctx.bicgstab_solve_eo(Ue, ee, kappa, r_min, 500)
        assert info["status"] == 0, info
    print("even-odd", dims, links, precision, "ok", flush=True)


if __name__ == "__main__":
    big = "--big" in sys.argv
    for precision in (32, 64):
        plain((4, 4, 4, 4), "haar", precision)
        plain((5, 7, 4, 6), "near_identity", precision)
        even_odd((4, 4, 4, 4), "haar", precision)
        even_odd((6, 6, 6, 6), "near_identity", precision)
        if big:
            plain((14, 14, 14, 14), "haar", precision)
            even_odd((14, 14, 14, 14), "haar", precision)
    print("sanitizer driver finished", flush=True)
