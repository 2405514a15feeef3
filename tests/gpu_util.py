"""Helpers of the -m gpu parity tests: move seeded canonical inputs to the device, call the C-ABI
binding, bring results back.  No arithmetic of the method lives here."""
import functools

import numpy as np

from paper_2111_14958_b200 import inputs


def np_complex(precision):
    return np.complex64 if precision == 32 else np.complex128


@functools.lru_cache(maxsize=4)
def config_fields(cfg_index, precision):
    """(U, eta) of a BASELINE config, generated in fp64 and rounded once to the run precision."""
    cfg = inputs.CONFIGS[cfg_index]
    return inputs.config_inputs(cfg, dtype=np_complex(precision))


def to_device(a):
    import torch

    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def to_host(t):
    return t.detach().cpu().numpy()


def apply_on_gpu(ctx, U, psi, kappa, dagger):
    """canonical numpy in -> wd_pack -> wd_apply -> wd_unpack -> canonical numpy out."""
    Un = ctx.wd_pack_gauge(to_device(U))
    pn = ctx.wd_pack_spinor(to_device(psi))
    out = ctx.wd_apply(Un, pn, kappa, dagger)
    return to_host(ctx.wd_unpack_spinor(out))


def solve_on_gpu(ctx, U, eta, kappa, r_min, max_iter):
    Un = ctx.wd_pack_gauge(to_device(U))
    en = ctx.wd_pack_spinor(to_device(eta))
    psi_n, info = ctx.cg_solve(Un, en, kappa, r_min, max_iter)
    return to_host(ctx.wd_unpack_spinor(psi_n)), info
