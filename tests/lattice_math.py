"""Independent mathematics used to PIN the oracle (tests only; never imported by oracle/ or the
CUDA package).  Nothing here calls the oracle's stencil: the dense matrix is assembled from
Kronecker blocks of covariant shift matrices, the free-field results are closed forms.

Reading C-1 / C-2 of SURVEY.md §8(c) (the paper only cites Wilson):
    D = 1 - kappa sum_mu [ (1 - gamma_mu) (x) T_mu + (1 + gamma_mu) (x) T_mu^dagger ],
    (T_mu psi)(x) = sigma+_mu(x) U_mu(x) psi(x + mu)      (covariant shift, unitary for unitary U).
"""
import numpy as np

I = 1j
# Reading C-2 (chiral basis); tests/test_oracle_pins.py::test_gamma_basis_extracted_from_oracle checks
# that the oracle realises exactly this set AND that it satisfies the Clifford algebra.
GAMMA = np.array([
    [[0, 0, 0, I], [0, 0, I, 0], [0, -I, 0, 0], [-I, 0, 0, 0]],
    [[0, 0, 0, -1], [0, 0, 1, 0], [0, 1, 0, 0], [-1, 0, 0, 0]],
    [[0, 0, I, 0], [0, 0, 0, -I], [-I, 0, 0, 0], [0, I, 0, 0]],
    [[0, 0, 1, 0], [0, 0, 0, 1], [1, 0, 0, 0], [0, 1, 0, 0]],
], dtype=np.complex128)
GAMMA5 = np.diag([1.0, 1.0, -1.0, -1.0]).astype(np.complex128)


def coords(dims):
    """(V, 4) integer coordinates of every site, x fastest."""
    lx, ly, lz, lt = dims
    s = np.arange(lx * ly * lz * lt)
    return np.stack([s % lx, (s // lx) % ly, (s // (lx * ly)) % lz, s // (lx * ly * lz)], axis=1)


def site_index(dims, xyzt):
    lx, ly, lz, _ = dims
    xyzt = np.asarray(xyzt)
    return xyzt[..., 0] + lx * (xyzt[..., 1] + ly * (xyzt[..., 2] + lz * xyzt[..., 3]))


def neighbour(dims, mu, step):
    """Site index of x + step*mu for every site (periodic wrap)."""
    c = coords(dims).copy()
    c[:, mu] = (c[:, mu] + step) % dims[mu]
    return site_index(dims, c)


def shift_matrix(dims, U, mu, bc_t):
    """Dense covariant shift T_mu, shape (V,3,V,3): T[x,a,x+mu,b] += sigma+(x) U_mu(x)[a,b]."""
    V = int(np.prod(dims))
    T = np.zeros((V, 3, V, 3), dtype=np.complex128)
    nb = neighbour(dims, mu, +1)
    xt = coords(dims)[:, 3]
    for x in range(V):
        sig = -1.0 if (mu == 3 and bc_t == -1 and xt[x] == dims[3] - 1) else 1.0
        T[x, :, nb[x], :] += sig * U[x, mu]
    return T


def dense_wilson(dims, U, kappa, bc_t=-1):
    """The 12V x 12V matrix of D, component index (s*4 + alpha)*3 + a."""
    V = int(np.prod(dims))
    M = np.eye(12 * V, dtype=np.complex128).reshape(V, 4, 3, V, 4, 3)
    one = np.eye(4)
    for mu in range(4):
        T = shift_matrix(dims, U, mu, bc_t)
        Tdag = np.conj(T.transpose(2, 3, 0, 1))
        M -= kappa * np.einsum("ij,xayb->xiayjb", one - GAMMA[mu], T)
        M -= kappa * np.einsum("ij,xayb->xiayjb", one + GAMMA[mu], Tdag)
    return M.reshape(12 * V, 12 * V)


def momenta(dims, n, bc_t=-1):
    """Lattice momentum for integer mode numbers n: 2 pi n/L, with (2n+1) pi/Lt in t if antiperiodic."""
    n = np.asarray(n, dtype=np.float64)
    p = 2.0 * np.pi * n / np.asarray(dims, dtype=np.float64)
    if bc_t == -1:
        p[..., 3] = (2.0 * n[..., 3] + 1.0) * np.pi / dims[3]
    return p


def plane_wave(dims, p, u):
    """psi(x) = u exp(i p.x), shape (V, 4, 3) for u of shape (4, 3)."""
    ph = np.exp(1j * (coords(dims) @ p))
    return ph[:, None, None] * u[None]


def free_dirac_symbol(p, kappa):
    """4x4 spin matrix D(p) = a + 2 i kappa sum_mu gamma_mu sin p_mu, a = 1 - 2 kappa sum cos p_mu (pin P3)."""
    a = 1.0 - 2.0 * kappa * np.sum(np.cos(p))
    return a * np.eye(4) + 2j * kappa * np.einsum("m,mij->ij", np.sin(p), GAMMA)


def free_dirac_inverse(p, kappa):
    """D(p)^-1 = [a - 2 i kappa gamma.sin p] / (a^2 + 4 kappa^2 sum sin^2 p) (pin P8)."""
    a = 1.0 - 2.0 * kappa * np.sum(np.cos(p))
    den = a * a + 4.0 * kappa * kappa * np.sum(np.sin(p) ** 2)
    return (a * np.eye(4) - 2j * kappa * np.einsum("m,mij->ij", np.sin(p), GAMMA)) / den


def free_point_propagator(dims, kappa, x0, u, bc_t=-1):
    """Exact psi with D psi = delta_{x,x0} u in the free field, by the inverse lattice Fourier sum.

    psi(x) = (1/V) sum_p exp(i p.(x - x0)) D(p)^-1 u.  FFT over the integer mode numbers; the
    half-integer t momenta of the antiperiodic case are a phase twist exp(i pi (t - t0)/Lt)."""
    lx, ly, lz, lt = dims
    nx = np.arange(lx)[None, None, None, :]
    ny = np.arange(ly)[None, None, :, None]
    nz = np.arange(lz)[None, :, None, None]
    nt = np.arange(lt)[:, None, None, None]
    px = 2 * np.pi * nx / lx
    py = 2 * np.pi * ny / ly
    pz = 2 * np.pi * nz / lz
    pt = (2 * nt + 1) * np.pi / lt if bc_t == -1 else 2 * np.pi * nt / lt
    a = 1.0 - 2.0 * kappa * (np.cos(px) + np.cos(py) + np.cos(pz) + np.cos(pt))
    s = [np.sin(px) + 0 * a, np.sin(py) + 0 * a, np.sin(pz) + 0 * a, np.sin(pt) + 0 * a]
    den = a * a + 4.0 * kappa * kappa * (s[0] ** 2 + s[1] ** 2 + s[2] ** 2 + s[3] ** 2)
    # Dinv(p) u, shape (Lt,Lz,Ly,Lx,4,3)
    gu = np.einsum("mij,ja->mia", GAMMA, u)
    field = a[..., None, None] * u[None, None, None, None]
    for mu in range(4):
        field = field - 2j * kappa * s[mu][..., None, None] * gu[mu][None, None, None, None]
    field = field / den[..., None, None]
    # phase exp(-i p.x0) in mode space (integer part), then inverse FFT (numpy ifft carries the 1/N).
    ph = np.exp(-1j * (px * x0[0] + py * x0[1] + pz * x0[2] + 2 * np.pi * nt * x0[3] / lt))
    field = field * ph[..., None, None]
    psi = np.fft.ifftn(field, axes=(0, 1, 2, 3))  # exp(+2 pi i n x / L) convention
    if bc_t == -1:
        t = np.arange(lt)[:, None, None, None]
        psi = psi * np.exp(1j * np.pi * (t - x0[3]) / lt)[..., None, None]
    return psi.reshape(lx * ly * lz * lt, 4, 3)


def free_solve(dims, kappa, eta, bc_t=-1):
    """Exact psi with D psi = eta in the free field (U = 1) for ANY source: Fourier transform, multiply every mode
    by the closed-form D(p)^-1 (pin P8), transform back.  The half-integer t momenta of the antiperiodic case are
    handled by untwisting the source with exp(-i pi t/Lt) and twisting the solution back."""
    lx, ly, lz, lt = dims
    f = np.asarray(eta, dtype=np.complex128).reshape(lt, lz, ly, lx, 4, 3)
    tw = np.exp(1j * np.pi * np.arange(lt) / lt)[:, None, None, None, None, None] if bc_t == -1 else 1.0
    ft = np.fft.fftn(f / tw, axes=(0, 1, 2, 3))
    nt = np.arange(lt)[:, None, None, None]
    pt = (2 * nt + 1) * np.pi / lt if bc_t == -1 else 2 * np.pi * nt / lt
    pz = 2 * np.pi * np.arange(lz)[None, :, None, None] / lz
    py = 2 * np.pi * np.arange(ly)[None, None, :, None] / ly
    px = 2 * np.pi * np.arange(lx)[None, None, None, :] / lx
    a = 1.0 - 2.0 * kappa * (np.cos(px) + np.cos(py) + np.cos(pz) + np.cos(pt))
    sn = [np.sin(px) + 0 * a, np.sin(py) + 0 * a, np.sin(pz) + 0 * a, np.sin(pt) + 0 * a]
    den = a * a + 4.0 * kappa * kappa * (sn[0] ** 2 + sn[1] ** 2 + sn[2] ** 2 + sn[3] ** 2)
    out = a[..., None, None] * ft
    for mu in range(4):
        out = out - 2j * kappa * sn[mu][..., None, None] * np.einsum("ij,...ja->...ia", GAMMA[mu], ft)
    out = out / den[..., None, None]
    psi = np.fft.ifftn(out, axes=(0, 1, 2, 3)) * tw
    return psi.reshape(lx * ly * lz * lt, 4, 3)


def gauge_rotate_links(dims, U, g):
    """U'_mu(x) = g(x) U_mu(x) g(x+mu)^dagger."""
    out = np.empty_like(U)
    for mu in range(4):
        gn = g[neighbour(dims, mu, +1)]
        out[:, mu] = np.einsum("xab,xbc,xdc->xad", g, U[:, mu], np.conj(gn))
    return out


def pure_gauge_links(dims, g):
    """U_mu(x) = g(x) g(x+mu)^dagger (gauge-equivalent to the free field)."""
    V = g.shape[0]
    one = np.broadcast_to(np.eye(3, dtype=np.complex128), (V, 4, 3, 3)).copy()
    return gauge_rotate_links(dims, one, g)


def per_site_rel_err(a, b):
    """max over sites of |a(x) - b(x)|_2 / |b(x)|_2 (reading G15) and the global relative L2 error."""
    a = np.asarray(a, dtype=np.complex128).reshape(-1, 12)
    b = np.asarray(b, dtype=np.complex128).reshape(-1, 12)
    num = np.linalg.norm(a - b, axis=1)
    den = np.linalg.norm(b, axis=1)
    return float(np.max(num / den)), float(np.linalg.norm(a - b) / np.linalg.norm(b))
