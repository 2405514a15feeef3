"""Pins of the CPU oracle against what the paper and the mathematics fix.

The paper prints no worked example (no matrix entries, residuals or iteration counts), so every
pin is brute force, a closed form or an invariant.  None of them calls the oracle to produce its
own expected value.  Runs with -m "not gpu".
"""
import numpy as np
import pytest

from paper_2111_14958_b200 import inputs
import lattice_math as lm

CFG_TEST = 900  # seeds for test-only lattices (distinct from BASELINE configs 0..4)


def rand_spinor(cfg, dims, field=inputs.FIELD_AUX):
    return inputs.source_field(cfg, dims, field=field)


def unit_gauge(dims):
    return inputs.gauge_field(0, dims, "unit")


# ---------------------------------------------------------------- P1: dense brute force
@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 3, 2, 4)])
@pytest.mark.parametrize("bc_t", [-1, +1])
def test_p1_dense_matrix(oracle, dims, bc_t):
    kappa = 0.12
    U = inputs.gauge_field(CFG_TEST + 1, dims, "haar")
    psi = rand_spinor(CFG_TEST + 1, dims)
    M = lm.dense_wilson(dims, U, kappa, bc_t)
    v = psi.reshape(-1)
    want = (M @ v).reshape(psi.shape)
    want_dag = (M.conj().T @ v).reshape(psi.shape)
    got = oracle.wd_apply(dims, U, psi, kappa, False, bc_t)
    got_dag = oracle.wd_apply(dims, U, psi, kappa, True, bc_t)
    assert np.max(np.abs(got - want)) < 1e-13
    assert np.max(np.abs(got_dag - want_dag)) < 1e-13
    # sampled-site entry point agrees with the dense rows too
    sites = np.array([0, 1, int(np.prod(dims)) - 1, 7])
    part = oracle.wd_apply_sites(dims, U, psi, kappa, sites, True, bc_t)
    assert np.max(np.abs(part - want_dag[sites])) < 1e-13


def test_p1_boundary_sign_matters(oracle):
    """Antiperiodic and periodic t differ exactly on the two boundary t-slices."""
    dims = (4, 3, 2, 4)
    U = inputs.gauge_field(CFG_TEST + 2, dims, "haar")
    psi = rand_spinor(CFG_TEST + 2, dims)
    a = oracle.wd_apply(dims, U, psi, 0.12, False, -1)
    p = oracle.wd_apply(dims, U, psi, 0.12, False, +1)
    t = lm.coords(dims)[:, 3]
    diff = np.abs(a - p).reshape(len(t), -1).max(axis=1)
    assert np.all(diff[(t != 0) & (t != dims[3] - 1)] == 0.0)
    assert np.all(diff[(t == 0) | (t == dims[3] - 1)] > 1e-3)


# ---------------------------------------------------------------- gamma basis (reading C-2)
def test_gamma_basis_extracted_from_oracle(oracle):
    """Extract gamma_mu from the oracle through the free-field symbol and check the algebra.

    With U = 1, periodic BC and a momentum along mu only, D psi = [a + 2 i kappa sin(p) gamma_mu] psi
    for psi = u exp(ipx) (PAPER.md:44 only states gamma5-hermiticity; the symbol is north_star's
    closed form).  The extracted matrices must be hermitian, square to one, anticommute, multiply to
    gamma5 = diag(1,1,-1,-1), and equal the table of reading C-2."""
    dims = (4, 4, 4, 4)
    kappa = 0.1
    U = unit_gauge(dims)
    got = []
    for mu in range(4):
        n = np.zeros(4)
        n[mu] = 1
        p = lm.momenta(dims, n, bc_t=+1)
        a = 1.0 - 2.0 * kappa * np.sum(np.cos(p))
        g = np.zeros((4, 4), dtype=np.complex128)
        for beta in range(4):
            u = np.zeros((4, 3), dtype=np.complex128)
            u[beta, 1] = 1.0
            psi = lm.plane_wave(dims, p, u)
            out = oracle.wd_apply(dims, U, psi, kappa, False, +1)
            col = out[0, :, 1] / psi[0, beta, 1]
            g[:, beta] = (col - a * np.eye(4)[:, beta]) / (2j * kappa * np.sin(p[mu]))
        got.append(g)
    got = np.array(got)
    for mu in range(4):
        assert np.allclose(got[mu], got[mu].conj().T, atol=1e-13)
        for nu in range(4):
            anti = got[mu] @ got[nu] + got[nu] @ got[mu]
            assert np.allclose(anti, 2.0 * (mu == nu) * np.eye(4), atol=1e-12)
    assert np.allclose(got[0] @ got[1] @ got[2] @ got[3], lm.GAMMA5, atol=1e-12)
    assert np.allclose(got, lm.GAMMA, atol=1e-13)


# ---------------------------------------------------------------- P2: gamma5-hermiticity
@pytest.mark.parametrize("links", ["haar", "near_identity"])
@pytest.mark.parametrize("bc_t", [-1, +1])
def test_p2_gamma5_hermiticity(oracle, links, bc_t):
    dims = (4, 6, 4, 8)
    kappa = 0.124
    U = inputs.gauge_field(CFG_TEST + 3, dims, links)
    psi = rand_spinor(CFG_TEST + 3, dims)
    chi = rand_spinor(CFG_TEST + 4, dims)
    g5 = np.array([1, 1, -1, -1.0])[None, :, None]
    ddag = oracle.wd_apply(dims, U, psi, kappa, True, bc_t)
    g5dg5 = g5 * oracle.wd_apply(dims, U, g5 * psi, kappa, False, bc_t)
    assert np.max(np.abs(ddag - g5dg5)) < 1e-13
    # <chi, D psi> = <D-dagger chi, psi>
    lhs = np.vdot(chi, oracle.wd_apply(dims, U, psi, kappa, False, bc_t))
    rhs = np.vdot(oracle.wd_apply(dims, U, chi, kappa, True, bc_t), psi)
    assert abs(lhs - rhs) < 1e-10 * abs(lhs)


def test_ddagger_hermitian_positive(oracle):
    """D D-dagger is 'hermitian by construction' and positive definite."""
    dims = (4, 4, 4, 4)
    kappa = 0.12
    U = inputs.gauge_field(CFG_TEST + 5, dims, "haar")
    psi = rand_spinor(CFG_TEST + 5, dims)
    chi = rand_spinor(CFG_TEST + 6, dims)

    def ddd(v):
        return oracle.wd_apply(dims, U, oracle.wd_apply(dims, U, v, kappa, True), kappa, False)

    a = np.vdot(chi, ddd(psi))
    b = np.conj(np.vdot(psi, ddd(chi)))
    assert abs(a - b) < 1e-10 * abs(a)
    e = np.vdot(psi, ddd(psi))
    assert e.real > 0 and abs(e.imag) < 1e-10 * e.real


# ---------------------------------------------------------------- P3: free-field plane waves
@pytest.mark.parametrize("bc_t", [-1, +1])
@pytest.mark.parametrize("dagger", [False, True])
def test_p3_free_field_symbol(oracle, bc_t, dagger):
    dims = (4, 3, 2, 4)
    kappa = 0.12
    U = unit_gauge(dims)
    rng = np.random.default_rng(5)
    for n in [(1, 2, 1, 3), (0, 0, 0, 0), (3, 1, 0, 2)]:
        p = lm.momenta(dims, np.array(n, dtype=float), bc_t)
        u = rng.standard_normal((4, 3)) + 1j * rng.standard_normal((4, 3))
        psi = lm.plane_wave(dims, p, u)
        sym = lm.free_dirac_symbol(p, kappa)
        if dagger:
            sym = sym.conj().T
        want = lm.plane_wave(dims, p, sym @ u)
        got = oracle.wd_apply(dims, U, psi, kappa, dagger, bc_t)
        assert np.max(np.abs(got - want)) < 1e-13


# ---------------------------------------------------------------- P4: gauge covariance
@pytest.mark.parametrize("dagger", [False, True])
def test_p4_gauge_covariance(oracle, dagger):
    dims = (4, 6, 4, 8)
    kappa = 0.124
    U = inputs.gauge_field(CFG_TEST + 7, dims, "haar")
    g = inputs.gauge_transform_field(CFG_TEST + 7, dims)
    psi = rand_spinor(CFG_TEST + 7, dims)
    Ug = lm.gauge_rotate_links(dims, U, g)
    psig = np.einsum("xab,xsb->xsa", g, psi)
    lhs = oracle.wd_apply(dims, Ug, psig, kappa, dagger, -1)
    rhs = np.einsum("xab,xsb->xsa", g, oracle.wd_apply(dims, U, psi, kappa, dagger, -1))
    assert np.max(np.abs(lhs - rhs)) < 1e-13


# ---------------------------------------------------------------- P5: per-direction unitarity
@pytest.mark.parametrize("mu", [0, 1, 2, 3])
@pytest.mark.parametrize("dagger", [False, True])
def test_p5_direction_pair_is_twice_unitary(oracle, mu, dagger):
    """H_mu = (1-g_mu) T_mu + (1+g_mu) T_mu^dagger satisfies |H_mu psi| = 2 |psi| for unitary links.
    A single direction is isolated by zeroing the links of the other three."""
    dims = (4, 3, 4, 5)
    kappa = 0.3
    U = inputs.gauge_field(CFG_TEST + 8, dims, "haar")
    Umu = np.zeros_like(U)
    Umu[:, mu] = U[:, mu]
    psi = rand_spinor(CFG_TEST + 8, dims)
    h = (psi - oracle.wd_apply(dims, Umu, psi, kappa, dagger, -1)) / kappa
    assert abs(np.linalg.norm(h) - 2.0 * np.linalg.norm(psi)) < 1e-12 * np.linalg.norm(psi)


def test_p5_singular_value_bounds(oracle):
    """Free periodic field attains |D psi|/|psi| = 1 - 8 kappa (p=0) and 1 + 8 kappa (p=pi)."""
    dims = (4, 4, 4, 4)
    kappa = 0.12
    U = unit_gauge(dims)
    u = np.zeros((4, 3), dtype=np.complex128)
    u[2, 0] = 1.0
    for n, val in [((0, 0, 0, 0), 1 - 8 * kappa), ((2, 2, 2, 2), 1 + 8 * kappa)]:
        psi = lm.plane_wave(dims, lm.momenta(dims, np.array(n, float), +1), u)
        out = oracle.wd_apply(dims, U, psi, kappa, False, +1)
        assert abs(np.linalg.norm(out) / np.linalg.norm(psi) - val) < 1e-13


# ---------------------------------------------------------------- P6: CG vs direct solve (2^4)
@pytest.mark.parametrize("bc_t", [-1, +1])
def test_p6_cg_matches_dense_solve(oracle, bc_t):
    dims = (2, 2, 2, 2)
    kappa = 0.12
    U = inputs.gauge_field(CFG_TEST + 9, dims, "haar")
    eta = inputs.source_field(CFG_TEST + 9, dims)
    M = lm.dense_wilson(dims, U, kappa, bc_t)
    exact = np.linalg.solve(M, eta.reshape(-1)).reshape(eta.shape)
    psi, info = oracle.cg_solve(dims, U, eta, kappa, 1e-12, 500, bc_t, history=True)
    assert info["converged"] and info["status"] == 0
    assert np.linalg.norm(psi - exact) < 1e-10 * np.linalg.norm(exact)
    # |psi_k - psi*| is monotonically non-increasing: CG on D D-dagger minimises exactly this.
    errs = []
    for k in range(0, info["iterations"] + 1):
        pk, ik = oracle.cg_solve(dims, U, eta, kappa, 1e-12, k, bc_t)
        assert ik["iterations"] == k
        errs.append(np.linalg.norm(pk - exact))
    errs = np.array(errs)
    assert np.all(errs[1:] <= errs[:-1] * (1 + 1e-9) + 1e-13)
    assert errs[0] == pytest.approx(np.linalg.norm(exact))  # psi0 = 0
    # the recursed residual history ends below tolerance and starts at <eta,eta>
    assert info["rr_history"][0] == pytest.approx(np.vdot(eta, eta).real, rel=1e-14)
    assert np.sqrt(info["rr_history"][-1] / info["rr_history"][0]) < 1e-12


def test_p6_alpha_uses_squared_norms(oracle):
    """Reading G1: one CG step from psi0=0 gives y1 = alpha eta with alpha = <eta,eta>/<D^dag eta, D^dag eta>,
    so psi after 1 iteration = alpha D-dagger eta.  Computed here from the dense matrix."""
    dims = (2, 2, 2, 2)
    kappa = 0.11
    U = inputs.gauge_field(CFG_TEST + 10, dims, "haar")
    eta = inputs.source_field(CFG_TEST + 10, dims)
    M = lm.dense_wilson(dims, U, kappa, -1)
    q = M.conj().T @ eta.reshape(-1)
    alpha = np.vdot(eta, eta).real / np.vdot(q, q).real
    psi, info = oracle.cg_solve(dims, U, eta, kappa, 1e-30, 1, -1)
    assert info["iterations"] == 1 and info["status"] == 1 and not info["converged"]
    assert np.linalg.norm(psi.reshape(-1) - alpha * q) < 1e-13 * np.linalg.norm(q)
    # two steps: check beta and the second alpha the same way
    r1 = eta.reshape(-1) - alpha * (M @ q)
    beta = np.vdot(r1, r1).real / np.vdot(eta, eta).real
    p1 = r1 + beta * eta.reshape(-1)
    q1 = M.conj().T @ p1
    alpha1 = np.vdot(r1, r1).real / np.vdot(q1, q1).real
    y2 = alpha * eta.reshape(-1) + alpha1 * p1
    psi2, _ = oracle.cg_solve(dims, U, eta, kappa, 1e-30, 2, -1)
    assert np.linalg.norm(psi2.reshape(-1) - M.conj().T @ y2) < 1e-12 * np.linalg.norm(q)


# ---------------------------------------------------------------- P7: finite termination
@pytest.mark.parametrize("bc_t,expected", [(+1, 5), (-1, 4)])
def test_p7_free_field_finite_termination(oracle, bc_t, expected):
    """On 2^4 with U=1, D D-dagger has exactly 5 (periodic t) / 4 (antiperiodic t) distinct eigenvalues,
    so CG terminates in that many iterations."""
    dims = (2, 2, 2, 2)
    kappa = 0.1
    U = unit_gauge(dims)
    M = lm.dense_wilson(dims, U, kappa, bc_t)
    ev = np.linalg.eigvalsh(M @ M.conj().T)
    assert len(np.unique(np.round(ev, 10))) == expected
    eta = inputs.source_field(CFG_TEST + 11, dims)
    psi, info = oracle.cg_solve(dims, U, eta, kappa, 1e-11, 50, bc_t)
    assert info["iterations"] == expected
    exact = np.linalg.solve(M, eta.reshape(-1)).reshape(eta.shape)
    assert np.linalg.norm(psi - exact) < 1e-10 * np.linalg.norm(exact)


def test_p7_kappa_zero_is_identity(oracle):
    dims = (4, 4, 4, 4)
    U = inputs.gauge_field(CFG_TEST + 12, dims, "haar")
    eta = inputs.source_field(CFG_TEST + 12, dims)
    psi, info = oracle.cg_solve(dims, U, eta, 0.0, 1e-12, 10)
    assert info["iterations"] == 1
    assert np.max(np.abs(psi - eta)) < 1e-14


def test_zero_source_and_max_iter(oracle):
    dims = (4, 4, 4, 4)
    U = inputs.gauge_field(CFG_TEST + 12, dims, "haar")
    eta = np.zeros((256, 4, 3), dtype=np.complex128)
    psi, info = oracle.cg_solve(dims, U, eta, 0.12, 1e-6, 10)
    assert info["iterations"] == 0 and info["converged"] and np.all(psi == 0)
    eta = inputs.source_field(CFG_TEST + 12, dims)
    psi, info = oracle.cg_solve(dims, U, eta, 0.12, 1e-6, 0)
    assert info["iterations"] == 0 and info["status"] == 1 and np.all(psi == 0)


# ---------------------------------------------------------------- P8: closed-form inverse
def test_p8_plane_wave_sum_inverse(oracle):
    """K plane waves with distinct |D(p)|^2: CG stops after exactly K iterations at the closed-form psi."""
    dims = (4, 6, 4, 8)
    kappa = 0.12
    U = unit_gauge(dims)
    rng = np.random.default_rng(11)
    eta = np.zeros((int(np.prod(dims)), 4, 3), dtype=np.complex128)
    exact = np.zeros_like(eta)
    modes = [(1, 2, 0, 3), (0, 1, 1, 0), (2, 5, 3, 6)]
    scal = set()
    for n in modes:
        p = lm.momenta(dims, np.array(n, float), -1)
        u = rng.standard_normal((4, 3)) + 1j * rng.standard_normal((4, 3))
        eta += lm.plane_wave(dims, p, u)
        exact += lm.plane_wave(dims, p, lm.free_dirac_inverse(p, kappa) @ u)
        scal.add(round(float(np.linalg.det(lm.free_dirac_symbol(p, kappa)).real), 9))
    assert len(scal) == len(modes)
    psi, info = oracle.cg_solve(dims, U, eta, kappa, 1e-11, 100, -1)
    assert info["iterations"] == len(modes)
    assert np.linalg.norm(psi - exact) < 1e-10 * np.linalg.norm(exact)


@pytest.mark.parametrize("bc_t", [-1, +1])
def test_p8_point_source_fourier_and_pure_gauge(oracle, bc_t):
    dims = (4, 6, 4, 8)
    kappa = 0.12
    V = int(np.prod(dims))
    x0 = (1, 4, 2, 5)
    s0 = int(lm.site_index(dims, np.array(x0)))
    rng = np.random.default_rng(3)
    u = rng.standard_normal((4, 3)) + 1j * rng.standard_normal((4, 3))
    exact_free = lm.free_point_propagator(dims, kappa, x0, u, bc_t)
    # the Fourier-sum propagator really inverts the free operator (independent check of the pin itself)
    eta = np.zeros((V, 4, 3), dtype=np.complex128)
    eta[s0] = u
    psi, info = oracle.cg_solve(dims, unit_gauge(dims), eta, kappa, 1e-12, 2000, bc_t)
    assert info["converged"] and info["iterations"] > 10
    assert np.linalg.norm(psi - exact_free) < 1e-9 * np.linalg.norm(exact_free)
    # pure-gauge extension: every link non-trivial, exact solution g(x) psi_free(x) for source g(x0) u
    g = inputs.gauge_transform_field(CFG_TEST + 13, dims)
    Ug = lm.pure_gauge_links(dims, g)
    assert np.max(np.abs(Ug[:, 0] - np.eye(3))) > 0.5
    eta_g = np.zeros_like(eta)
    eta_g[s0] = g[s0] @ u.T @ np.eye(3) if False else np.einsum("ab,sb->sa", g[s0], u)
    psi_g, info_g = oracle.cg_solve(dims, Ug, eta_g, kappa, 1e-12, 2000, bc_t)
    want = np.einsum("xab,xsb->xsa", g, exact_free)
    assert info_g["iterations"] == pytest.approx(info["iterations"], abs=2)
    assert np.linalg.norm(psi_g - want) < 1e-9 * np.linalg.norm(want)


# ---------------------------------------------------------------- P9 / P10
def test_p9_norm(oracle):
    cfg = inputs.CONFIGS[1]
    eta = inputs.source_field(cfg.index, cfg.dims)
    n2 = oracle.norm2(eta)
    assert n2 == pytest.approx(float(np.sum(np.abs(eta) ** 2)), rel=1e-13)
    # re, im each N(0,1): <eta,eta> ~ 2 * 12 V within 5 sigma (chi^2 with 24V dof)
    dof = 24 * cfg.volume
    assert abs(n2 - dof) < 5 * np.sqrt(2 * dof)


def test_p10_true_vs_recursed_residual(oracle):
    cfg = inputs.CONFIGS[0]
    U, eta = inputs.config_inputs(cfg)
    psi, info = oracle.cg_solve(cfg.dims, U, eta, cfg.kappa, 1e-10, 1000)
    assert info["converged"]
    true = oracle.true_residual(cfg.dims, U, eta, psi, cfg.kappa)
    assert abs(true - info["rel_residual"]) < 1e-12
    assert true < 1e-10


# ---------------------------------------------------------------- P11: the paper's COO route
def test_p11_coo_spmv(oracle):
    """Alg. COO of PAPER.md:52-54 on the matrix assembled from the definition: every row has
    1 + 8*2*3 = 49 non-zeros, N_NZ = 588 V, and out[Row[k]] += Val[k]*in[Col[k]] equals the stencil."""
    dims = (3, 4, 3, 4)
    V = int(np.prod(dims))
    kappa = 0.12
    U = inputs.gauge_field(CFG_TEST + 14, dims, "haar")
    psi = rand_spinor(CFG_TEST + 14, dims)
    M = lm.dense_wilson(dims, U, kappa, -1)
    row, col = np.nonzero(M)
    val = M[row, col]
    assert len(val) == 588 * V
    assert np.all(np.bincount(row, minlength=12 * V) == 49)
    out = np.zeros(12 * V, dtype=np.complex128)
    np.add.at(out, row, val * psi.reshape(-1)[col])
    got = oracle.wd_apply(dims, U, psi, kappa, False, -1)
    assert np.max(np.abs(got.reshape(-1) - out)) < 1e-13


# ---------------------------------------------------------------- BiCGSTAB (reading B1)
@pytest.mark.parametrize("bc_t", [-1, +1])
def test_bp1_bicgstab_matches_dense_solve(oracle, bc_t):
    dims = (2, 2, 2, 2)
    kappa = 0.12
    U = inputs.gauge_field(CFG_TEST + 20, dims, "haar")
    eta = inputs.source_field(CFG_TEST + 20, dims)
    M = lm.dense_wilson(dims, U, kappa, bc_t)
    exact = np.linalg.solve(M, eta.reshape(-1)).reshape(eta.shape)
    psi, info = oracle.bicgstab_solve(dims, U, eta, kappa, 1e-12, 500, bc_t, history=True)
    assert info["converged"] and info["status"] == 0
    assert np.linalg.norm(psi - exact) < 1e-10 * np.linalg.norm(exact)
    assert info["rr_history"][0] == pytest.approx(np.vdot(eta, eta).real, rel=1e-14)
    # residual identity: the recursed r equals eta - D psi
    assert abs(oracle.true_residual(dims, U, eta, psi, kappa, bc_t) - info["rel_residual"]) < 1e-12


def test_bp2_bicgstab_first_iterates_from_dense_matrix(oracle):
    """The listing of reading B1 retyped with the dense matrix (complex alpha, omega, beta; <a,b> = sum conj(a) b):
    pins the inner-product conjugation, the order of the updates and the beta formula."""
    dims = (2, 2, 2, 2)
    kappa = 0.11
    U = inputs.gauge_field(CFG_TEST + 21, dims, "haar")
    eta = inputs.source_field(CFG_TEST + 21, dims)
    M = lm.dense_wilson(dims, U, kappa, -1)
    b = eta.reshape(-1)
    x = np.zeros_like(b)
    r = b.copy()
    rhat = b.copy()
    p = r.copy()
    rho = np.vdot(rhat, r)
    for k in range(1, 4):
        v = M @ p
        alpha = rho / np.vdot(rhat, v)
        s = r - alpha * v
        t = M @ s
        omega = np.vdot(t, s) / np.vdot(t, t)
        x = x + alpha * p + omega * s
        r = s - omega * t
        rho_new = np.vdot(rhat, r)
        beta = (rho_new / rho) * (alpha / omega)
        p = r + beta * (p - omega * v)
        rho = rho_new
        psi, info = oracle.bicgstab_solve(dims, U, eta, kappa, 1e-30, k, -1, history=True)
        assert info["iterations"] == k and info["status"] == 1
        assert np.linalg.norm(psi.reshape(-1) - x) < 1e-12 * np.linalg.norm(x)
        assert info["rr_history"][k] == pytest.approx(np.vdot(r, r).real, rel=1e-9)
    # alpha and omega are genuinely complex here (a real-arithmetic shortcut would fail above)
    assert abs(alpha.imag) > 1e-6 * abs(alpha) or abs(omega.imag) > 1e-6 * abs(omega)


def test_bp3_bicgstab_finite_termination(oracle):
    """Free field, one plane wave: D acts as the 4x4 symbol a + 2 i kappa gamma.sin p, a normal matrix with two
    distinct eigenvalues a +- 2 i kappa |sin p| -> BiCGSTAB is exact after 2 iterations; kappa = 0 -> after 1."""
    dims = (4, 6, 4, 8)
    kappa = 0.12
    U = unit_gauge(dims)
    rng = np.random.default_rng(5)
    p = lm.momenta(dims, np.array((1, 2, 0, 3), float), -1)
    u = rng.standard_normal((4, 3)) + 1j * rng.standard_normal((4, 3))
    ev = np.linalg.eigvals(lm.free_dirac_symbol(p, kappa))
    assert len(np.unique(np.round(ev, 10))) == 2
    eta = lm.plane_wave(dims, p, u)
    psi, info = oracle.bicgstab_solve(dims, U, eta, kappa, 1e-11, 50, -1)
    assert info["iterations"] == 2 and info["converged"]
    exact = lm.plane_wave(dims, p, lm.free_dirac_inverse(p, kappa) @ u)
    assert np.linalg.norm(psi - exact) < 1e-10 * np.linalg.norm(exact)
    Uh = inputs.gauge_field(CFG_TEST + 22, dims, "haar")
    src = inputs.source_field(CFG_TEST + 22, dims)
    psi, info = oracle.bicgstab_solve(dims, Uh, src, 0.0, 1e-12, 10)
    assert info["iterations"] == 1 and np.max(np.abs(psi - src)) < 1e-14


def test_bp4_bicgstab_point_source_and_edge_cases(oracle):
    dims = (4, 6, 4, 8)
    kappa = 0.12
    V = int(np.prod(dims))
    rng = np.random.default_rng(3)
    # one point source in the free field: alpha = 1 (unit diagonal), s = kappa H delta, and
    # rho' = <delta, r1> = omega kappa^2 (H^2 delta)(x0) = 0 because (1 - gamma_mu)(1 + gamma_mu) = 0:
    # a genuine BiCGSTAB breakdown after exactly one iteration, reported as status 2.
    x0 = (1, 4, 2, 5)
    u = rng.standard_normal((4, 3)) + 1j * rng.standard_normal((4, 3))
    eta = np.zeros((V, 4, 3), dtype=np.complex128)
    eta[int(lm.site_index(dims, np.array(x0)))] = u
    psi, info = oracle.bicgstab_solve(dims, unit_gauge(dims), eta, kappa, 1e-12, 2000, -1)
    assert info["status"] == 2 and info["iterations"] == 1 and not info["converged"]
    # a Gaussian source (no such symmetry): exact solution mode by mode with the closed-form D(p)^-1 (pin P8);
    # the Fourier route itself is checked against the point-source propagator first
    chk = lm.free_solve(dims, kappa, eta, -1)
    assert np.linalg.norm(chk - lm.free_point_propagator(dims, kappa, x0, u, -1)) < 1e-12 * np.linalg.norm(chk)
    eta = inputs.source_field(CFG_TEST + 23, dims)
    exact = lm.free_solve(dims, kappa, eta, -1)
    psi, info = oracle.bicgstab_solve(dims, unit_gauge(dims), eta, kappa, 1e-12, 2000, -1)
    assert info["converged"] and info["iterations"] > 5
    assert np.linalg.norm(psi - exact) < 1e-9 * np.linalg.norm(exact)
    # the same solution as the CG route on a Haar field
    cfg = inputs.CONFIGS[0]
    Uc, ec = inputs.config_inputs(cfg)
    pb, ib = oracle.bicgstab_solve(cfg.dims, Uc, ec, cfg.kappa, 1e-11, 1000)
    pc, ic = oracle.cg_solve(cfg.dims, Uc, ec, cfg.kappa, 1e-11, 1000)
    assert ib["converged"] and ic["converged"] and ib["iterations"] < ic["iterations"]
    assert np.linalg.norm(pb - pc) < 1e-9 * np.linalg.norm(pc)
    # eta = 0 and max_iter = 0
    z, iz = oracle.bicgstab_solve(cfg.dims, Uc, np.zeros_like(ec), cfg.kappa, 1e-6, 10)
    assert iz["iterations"] == 0 and iz["converged"] and np.all(z == 0)
    z, iz = oracle.bicgstab_solve(cfg.dims, Uc, ec, cfg.kappa, 1e-6, 0)
    assert iz["iterations"] == 0 and iz["status"] == 1 and np.all(z == 0)


# ---------------------------------------------------------------- COO assembly
@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (3, 4, 3, 4)])
@pytest.mark.parametrize("dagger", [False, True])
def test_cp1_coo_assembly_is_the_dense_matrix(oracle, dims, dagger):
    """The assembled (Val, Row, Col) scattered into a dense array equals the Kronecker-block matrix (its
    conjugate transpose for dagger); 49 entries per row, N_NZ = 588 V (duplicates on 2^4 are summed)."""
    V = int(np.prod(dims))
    kappa = 0.12
    U = inputs.gauge_field(CFG_TEST + 30, dims, "haar")
    val, row, col = oracle.coo_assemble(dims, U, kappa, dagger, -1)
    assert val.size == 588 * V and np.all(np.bincount(row, minlength=12 * V) == 49)
    assert np.all(row[::49] == np.arange(12 * V)) and np.all(col[::49] == np.arange(12 * V)) and np.all(val[::49] == 1)
    M = lm.dense_wilson(dims, U, kappa, -1)
    if dagger:
        M = M.conj().T
    A = np.zeros_like(M)
    np.add.at(A, (row, col), val)
    assert np.max(np.abs(A - M)) < 1e-14
    if min(dims) > 2:   # all (row, col) pairs distinct
        assert len(set(zip(row.tolist(), col.tolist()))) == val.size


def test_cp2_coo_spmv_equals_stencil(oracle):
    dims = (4, 6, 4, 8)
    kappa = 0.124
    U = inputs.gauge_field(CFG_TEST + 31, dims, "near_identity")
    psi = rand_spinor(CFG_TEST + 31, dims)
    for dagger in (False, True):
        val, row, col = oracle.coo_assemble(dims, U, kappa, dagger, -1)
        got = oracle.coo_spmv(val, row, col, psi)
        want = oracle.wd_apply(dims, U, psi, kappa, dagger, -1)
        assert np.max(np.abs(got - want)) < 1e-13
    # numpy's scatter-add on the same arrays (an independent execution of the paper's loop)
    ref = np.zeros(psi.size, dtype=np.complex128)
    np.add.at(ref, row, val * psi.reshape(-1)[col])
    assert np.max(np.abs(ref - got.reshape(-1))) < 1e-13


# ---------------------------------------------------------------- even-odd preconditioned CG (reading E1)
def _parity(dims):
    return lm.coords(dims).sum(axis=1) & 1


def _dense_blocks(dims, U, kappa, bc_t):
    """M_ee, M_eo, M_oe, M_oo of the Kronecker-built dense D, and the component index sets of the two parities"""
    M = lm.dense_wilson(dims, U, kappa, bc_t)
    par = np.repeat(_parity(dims), 12)
    e, o = np.nonzero(par == 0)[0], np.nonzero(par == 1)[0]
    return M, e, o


@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 2, 2, 4)])
@pytest.mark.parametrize("bc_t", [-1, +1])
def test_ep1_schur_operator_is_the_dense_schur_complement(oracle, dims, bc_t):
    kappa = 0.12
    U = inputs.gauge_field(CFG_TEST + 40, dims, "haar")
    v = rand_spinor(CFG_TEST + 40, dims)
    M, e, o = _dense_blocks(dims, U, kappa, bc_t)
    assert np.allclose(M[np.ix_(e, e)], np.eye(e.size)) and np.allclose(M[np.ix_(o, o)], np.eye(o.size))
    S = M[np.ix_(e, e)] - M[np.ix_(e, o)] @ M[np.ix_(o, e)]      # D_ee - D_eo D_oo^-1 D_oe with D_oo = 1
    for dagger, A in ((False, S), (True, S.conj().T)):
        got = oracle.schur_apply(dims, U, v, kappa, dagger, bc_t).reshape(-1)
        assert np.max(np.abs(got[e] - A @ v.reshape(-1)[e])) < 1e-13
        assert not got[o].any()


@pytest.mark.parametrize("bc_t", [-1, +1])
def test_ep2_eo_cg_matches_dense_solve_and_plain_cg(oracle, bc_t):
    dims = (4, 2, 2, 4)
    kappa = 0.12
    U = inputs.gauge_field(CFG_TEST + 41, dims, "haar")
    eta = inputs.source_field(CFG_TEST + 41, dims)
    M = lm.dense_wilson(dims, U, kappa, bc_t)
    exact = np.linalg.solve(M, eta.reshape(-1)).reshape(eta.shape)
    psi, info = oracle.cg_solve_eo(dims, U, eta, kappa, 1e-12, 500, bc_t, history=True)
    assert info["converged"] and info["status"] == 0
    assert np.linalg.norm(psi - exact) < 1e-10 * np.linalg.norm(exact)
    # the recursed residual IS the true residual of the full system (its odd rows vanish identically)
    assert abs(oracle.true_residual(dims, U, eta, psi, kappa, bc_t) - info["rel_residual"]) < 1e-12
    r_full = (eta - oracle.wd_apply(dims, U, psi, kappa, False, bc_t)).reshape(-1, 12)
    assert np.max(np.abs(r_full[_parity(dims) == 1])) < 1e-13
    # first history entry: <etahat, etahat> with etahat = eta_e - M_eo eta_o from the dense blocks
    _, e, o = _dense_blocks(dims, U, kappa, bc_t)
    etahat = eta.reshape(-1)[e] - M[np.ix_(e, o)] @ eta.reshape(-1)[o]
    assert info["rr_history"][0] == pytest.approx(np.vdot(etahat, etahat).real, rel=1e-13)
    assert info["eta_norm2"] == pytest.approx(np.vdot(eta, eta).real, rel=1e-13)
    # same solution as the unpreconditioned recurrence, in fewer iterations
    psi_p, info_p = oracle.cg_solve(dims, U, eta, kappa, 1e-12, 500, bc_t)
    assert np.linalg.norm(psi - psi_p) < 1e-10 * np.linalg.norm(psi_p)
    assert info["iterations"] < info_p["iterations"]


def test_ep3_eo_cg_first_step_and_finite_termination(oracle):
    """one step retyped from the dense Schur complement (pins alpha, the order Mhat-dagger then Mhat, and the
    reconstruction of psi_o); free field on 2^4: as many iterations as Mhat Mhat-dagger has distinct eigenvalues"""
    dims = (2, 2, 2, 2)
    kappa = 0.11
    U = inputs.gauge_field(CFG_TEST + 42, dims, "haar")
    eta = inputs.source_field(CFG_TEST + 42, dims)
    M, e, o = _dense_blocks(dims, U, kappa, -1)
    S = M[np.ix_(e, e)] - M[np.ix_(e, o)] @ M[np.ix_(o, e)]
    b = eta.reshape(-1)
    etahat = b[e] - M[np.ix_(e, o)] @ b[o]
    q = S.conj().T @ etahat
    alpha = np.vdot(etahat, etahat).real / np.vdot(q, q).real
    psi_e = S.conj().T @ (alpha * etahat)
    want = np.zeros_like(b)
    want[e] = psi_e
    want[o] = b[o] - M[np.ix_(o, e)] @ psi_e
    psi, info = oracle.cg_solve_eo(dims, U, eta, kappa, 1e-30, 1, -1)
    assert info["iterations"] == 1 and info["status"] == 1
    assert np.linalg.norm(psi.reshape(-1) - want) < 1e-13 * np.linalg.norm(want)
    Uf = unit_gauge(dims)
    for bc_t in (-1, +1):
        Mf, e, o = _dense_blocks(dims, Uf, 0.1, bc_t)
        Sf = Mf[np.ix_(e, e)] - Mf[np.ix_(e, o)] @ Mf[np.ix_(o, e)]
        n_ev = len(np.unique(np.round(np.linalg.eigvalsh(Sf @ Sf.conj().T), 10)))
        psi, info = oracle.cg_solve_eo(dims, Uf, eta, 0.1, 1e-11, 50, bc_t)
        assert info["iterations"] == n_ev and info["converged"]
        exact = np.linalg.solve(Mf, eta.reshape(-1)).reshape(eta.shape)
        assert np.linalg.norm(psi - exact) < 1e-10 * np.linalg.norm(exact)


def test_ep4_eo_cg_baseline_configs_and_edge_cases(oracle):
    for ci in (0, 1):
        cfg = inputs.CONFIGS[ci]
        U, eta = inputs.config_inputs(cfg)
        pe, ie = oracle.cg_solve_eo(cfg.dims, U, eta, cfg.kappa, 1e-10, cfg.max_iter, cfg.bc_t)
        pp, ip = oracle.cg_solve(cfg.dims, U, eta, cfg.kappa, 1e-10, cfg.max_iter, cfg.bc_t)
        assert ie["converged"] and ie["iterations"] < 0.7 * ip["iterations"]
        assert np.linalg.norm(pe - pp) < 1e-8 * np.linalg.norm(pp)
        assert oracle.true_residual(cfg.dims, U, eta, pe, cfg.kappa, cfg.bc_t) < 1e-10
    z, iz = oracle.cg_solve_eo(cfg.dims, U, np.zeros_like(eta), cfg.kappa, 1e-6, 10)
    assert iz["iterations"] == 0 and iz["converged"] and not z.any()
    # max_iter = 0: psi_e = 0 and psi_o = eta_o (the exact odd rows for psi_e = 0)
    z, iz = oracle.cg_solve_eo(cfg.dims, U, eta, cfg.kappa, 1e-6, 0)
    par = _parity(cfg.dims)
    assert iz["iterations"] == 0 and iz["status"] == 1 and not z[par == 0].any() and np.array_equal(z[par == 1], eta[par == 1])
    with pytest.raises(RuntimeError):
        oracle.cg_solve_eo((4, 3, 4, 4), U[:192], eta[:192], 0.1, 1e-6, 10)   # odd extent


# ---------------------------------------------------------------- even-odd preconditioned BiCGSTAB (readings E1 + B1 = EB1)
@pytest.mark.parametrize("bc_t", [-1, +1])
def test_ebp1_eo_bicgstab_matches_dense_solve(oracle, bc_t):
    dims = (4, 2, 2, 4)
    kappa = 0.12
    U = inputs.gauge_field(CFG_TEST + 50, dims, "haar")
    eta = inputs.source_field(CFG_TEST + 50, dims)
    M, e, o = _dense_blocks(dims, U, kappa, bc_t)
    exact = np.linalg.solve(M, eta.reshape(-1)).reshape(eta.shape)
    psi, info = oracle.bicgstab_solve_eo(dims, U, eta, kappa, 1e-12, 500, bc_t, history=True)
    assert info["converged"] and info["status"] == 0
    assert np.linalg.norm(psi - exact) < 1e-10 * np.linalg.norm(exact)
    # the recursed residual is the true residual of the FULL system, whose odd rows vanish identically
    assert abs(oracle.true_residual(dims, U, eta, psi, kappa, bc_t) - info["rel_residual"]) < 1e-12
    r_full = (eta - oracle.wd_apply(dims, U, psi, kappa, False, bc_t)).reshape(-1, 12)
    assert np.max(np.abs(r_full[_parity(dims) == 1])) < 1e-13
    etahat = eta.reshape(-1)[e] - M[np.ix_(e, o)] @ eta.reshape(-1)[o]
    assert info["rr_history"][0] == pytest.approx(np.vdot(etahat, etahat).real, rel=1e-13)
    assert info["eta_norm2"] == pytest.approx(np.vdot(eta, eta).real, rel=1e-13)


def test_ebp2_eo_bicgstab_first_iterates_from_dense_schur_complement(oracle):
    """The listing of reading B1 retyped on the dense Schur complement of the Kronecker-built matrix, followed by the
    odd-site reconstruction from the dense off-diagonal block: pins that the iteration runs on Mhat (not Mhat-dagger,
    not D), the shadow residual etahat, the complex scalars and psi_o."""
    dims = (2, 2, 2, 2)
    kappa = 0.11
    U = inputs.gauge_field(CFG_TEST + 51, dims, "haar")
    eta = inputs.source_field(CFG_TEST + 51, dims)
    M, e, o = _dense_blocks(dims, U, kappa, -1)
    S = M[np.ix_(e, e)] - M[np.ix_(e, o)] @ M[np.ix_(o, e)]
    b = eta.reshape(-1)
    etahat = b[e] - M[np.ix_(e, o)] @ b[o]
    x = np.zeros_like(etahat)
    r = etahat.copy()
    rhat = etahat.copy()
    p = r.copy()
    rho = np.vdot(rhat, r)
    for k in range(1, 4):
        v = S @ p
        alpha = rho / np.vdot(rhat, v)
        s = r - alpha * v
        t = S @ s
        omega = np.vdot(t, s) / np.vdot(t, t)
        x = x + alpha * p + omega * s
        r = s - omega * t
        rho_new = np.vdot(rhat, r)
        beta = (rho_new / rho) * (alpha / omega)
        p = r + beta * (p - omega * v)
        rho = rho_new
        want = np.zeros_like(b)
        want[e] = x
        want[o] = b[o] - M[np.ix_(o, e)] @ x
        psi, info = oracle.bicgstab_solve_eo(dims, U, eta, kappa, 1e-30, k, -1, history=True)
        assert info["iterations"] == k and info["status"] == 1
        assert np.linalg.norm(psi.reshape(-1) - want) < 1e-12 * np.linalg.norm(want)
        assert info["rr_history"][k] == pytest.approx(np.vdot(r, r).real, rel=1e-9)
    assert abs(alpha.imag) > 1e-6 * abs(alpha) or abs(omega.imag) > 1e-6 * abs(omega)
    # Mhat is not normal here, so a solver on Mhat-dagger would give different iterates
    assert np.linalg.norm(S @ S.conj().T - S.conj().T @ S) > 1e-6


def test_ebp3_eo_bicgstab_special_cases_and_other_solvers(oracle):
    # kappa = 0: Mhat = 1, one iteration, psi = eta
    dims = (4, 6, 4, 8)
    Uh = inputs.gauge_field(CFG_TEST + 52, dims, "haar")
    src = inputs.source_field(CFG_TEST + 52, dims)
    psi, info = oracle.bicgstab_solve_eo(dims, Uh, src, 0.0, 1e-12, 10)
    assert info["iterations"] == 1 and info["converged"] and np.max(np.abs(psi - src)) < 1e-14
    # free field, Gaussian source: exact solution mode by mode with the closed-form D(p)^-1 (pin P8)
    kappa = 0.12
    exact = lm.free_solve(dims, kappa, src, -1)
    psi, info = oracle.bicgstab_solve_eo(dims, unit_gauge(dims), src, kappa, 1e-12, 2000, -1)
    assert info["converged"] and np.linalg.norm(psi - exact) < 1e-9 * np.linalg.norm(exact)
    # BASELINE configs 0, 1: same solution as the plain CG, fewer iterations than the plain BiCGSTAB and the even-odd CG
    for ci in (0, 1):
        cfg = inputs.CONFIGS[ci]
        U, eta = inputs.config_inputs(cfg)
        pe, ie = oracle.bicgstab_solve_eo(cfg.dims, U, eta, cfg.kappa, 1e-10, cfg.max_iter, cfg.bc_t)
        pb, ib = oracle.bicgstab_solve(cfg.dims, U, eta, cfg.kappa, 1e-10, cfg.max_iter, cfg.bc_t)
        pc, ic = oracle.cg_solve_eo(cfg.dims, U, eta, cfg.kappa, 1e-10, cfg.max_iter, cfg.bc_t)
        pp, ip = oracle.cg_solve(cfg.dims, U, eta, cfg.kappa, 1e-10, cfg.max_iter, cfg.bc_t)
        assert ie["converged"] and ie["iterations"] < ib["iterations"] and ie["iterations"] < ic["iterations"]
        assert np.linalg.norm(pe - pp) < 1e-8 * np.linalg.norm(pp)
        assert oracle.true_residual(cfg.dims, U, eta, pe, cfg.kappa, cfg.bc_t) < 1e-10
    z, iz = oracle.bicgstab_solve_eo(cfg.dims, U, np.zeros_like(eta), cfg.kappa, 1e-6, 10)
    assert iz["iterations"] == 0 and iz["converged"] and not z.any()
    z, iz = oracle.bicgstab_solve_eo(cfg.dims, U, eta, cfg.kappa, 1e-6, 0)
    par = _parity(cfg.dims)
    assert iz["iterations"] == 0 and iz["status"] == 1 and not z[par == 0].any() and np.array_equal(z[par == 1], eta[par == 1])
    with pytest.raises(RuntimeError):
        oracle.bicgstab_solve_eo((4, 3, 4, 4), U[:192], eta[:192], 0.1, 1e-6, 10)   # odd extent
