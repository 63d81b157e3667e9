"""Pins of the CPU oracle against what theory fixes (BASELINE.json north_star).

None of these compares the oracle with itself or with the CUDA path: closed forms, algebraic
invariants, and an independently assembled dense matrix (tests/dense_bruteforce.py).
"""
import os

import numpy as np
import pytest

from paper_2510_26313_b200 import inputs
from tests import dense_bruteforce as dbf

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
DIMS = (4, 4, 4, 8)


def lex_coords(dims):
    Lx, Ly, Lz, Lt = dims
    t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    return x, y, z, t


def vdot(a, b):
    return np.vdot(a.ravel(), b.ravel())


def rel(a, b):
    return np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel())


# ------------------------------------------------------------------ gamma matrices
def test_gamma_algebra(oracle_lib):
    g = [oracle_lib.gamma(mu) for mu in range(4)]
    for mu in range(4):
        assert np.array_equal(g[mu], g[mu].conj().T)
        for nu in range(4):
            anti = g[mu] @ g[nu] + g[nu] @ g[mu]
            assert np.allclose(anti, 2.0 * np.eye(4) * (mu == nu), atol=0)
    assert np.array_equal(oracle_lib.gamma(5), np.diag([1, 1, -1, -1]).astype(complex))
    assert np.array_equal(g[0] @ g[1] @ g[2] @ g[3], np.diag([1, 1, -1, -1]).astype(complex))
    assert np.array_equal(oracle_lib.sigma(0, 1), np.diag([1, -1, 1, -1]).astype(complex))
    for mu in range(4):          # table of SURVEY 8(c.1) step 2, retyped in dense_bruteforce.GAMMA
        assert np.array_equal(g[mu], dbf.GAMMA[mu])
    for mu in range(4):
        for nu in range(mu + 1, 4):
            s = oracle_lib.sigma(mu, nu)
            assert np.array_equal(s, s.conj().T)
            assert np.all(s[:2, 2:] == 0) and np.all(s[2:, :2] == 0)   # block-diagonal in chirality


# ------------------------------------------------------------------ inputs recipe
def test_links_are_su3_and_third_row_rule():
    U = inputs.make_links(DIMS, 1000, 0.3).reshape(-1, 3, 3)
    eye = np.eye(3)[None]
    assert np.abs(U @ U.conj().transpose(0, 2, 1) - eye).max() < 1e-14
    assert np.abs(np.linalg.det(U) - 1).max() < 1e-14
    assert np.abs(U[:, 2] - np.conj(np.cross(U[:, 0], U[:, 1]))).max() == 0
    # counter-based: regenerating one element from its index reproduces it
    U2 = inputs.make_links(DIMS, 1000, 0.3)
    assert np.array_equal(U2.reshape(-1, 3, 3), U)
    assert not np.array_equal(inputs.make_links(DIMS, 1001, 0.3).reshape(-1, 3, 3), U)


def test_cgauss_moments():
    z = inputs.cgauss(7, 2, np.arange(400000))
    assert abs(z.mean()) < 5e-3
    assert abs(np.mean(np.abs(z) ** 2) - 1.0) < 5e-3        # CN(0,1): E|z|^2 = 1 (reading #2)
    assert abs(np.mean(z.real ** 2) - 0.5) < 5e-3 and abs(np.mean(z.imag ** 2) - 0.5) < 5e-3
    assert abs(np.mean(z.real * z.imag)) < 5e-3


def test_laph_sources_structure():
    dims = (4, 4, 4, 8)
    b = inputs.laph_sources(dims, 8, 2, 2001)
    for k in range(8):
        t0 = (k // 4) * 4
        nz = np.nonzero(np.abs(b[k]).sum(axis=(1, 2, 3, 5)))  # timeslices, spins with support
        assert set(nz[0]) == {t0} and set(nz[1]) == {k % 4}
        assert abs(np.sum(np.abs(b[k]) ** 2) - 1.0) < 1e-14
    assert np.array_equal(b[0, 0, :, :, :, 0], b[1, 0, :, :, :, 1])    # one colour field per timeslice
    assert not np.array_equal(b[0, 0, :, :, :, 0], b[4, 4, :, :, :, 0])


# ------------------------------------------------------------------ free field (hop + boundary conditions)
def plane_wave(dims, n, u, theta=None):
    x, y, z, t = lex_coords(dims)
    p = [2 * np.pi * n[0] / dims[0], 2 * np.pi * n[1] / dims[1], 2 * np.pi * n[2] / dims[2],
         2 * np.pi * (n[3] + 0.5) / dims[3]]
    phase = np.exp(1j * (p[0] * x + p[1] * y + p[2] * z + p[3] * t))
    return phase[..., None, None] * u[None, None, None, None], np.array(p)


def load_golden_free_field():
    rows = []
    with open(os.path.join(GOLDEN, "free_field_4x4x4x8_kappa0p12.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            v = line.split()
            rows.append((tuple(int(q) for q in v[:4]), float(v[4]), float(v[5]), float(v[6])))
    return rows


@pytest.mark.parametrize("csw", [0.0, 1.0, 1.7])
def test_free_field_closed_form(oracle_lib, csw):
    kappa = 0.12
    U = inputs.unit_links(DIMS)
    A = oracle_lib.clover(DIMS, U, kappa, csw)
    assert np.array_equal(A.reshape(-1, 12, 12), np.broadcast_to(np.eye(12), (512, 12, 12)))  # A = 1 for any c_sw
    rng = np.random.default_rng(5)
    for n, a_ref, b_ref, n2_ref in load_golden_free_field() + [((3, 1, 2, 5), None, None, None), ((0, 3, 0, 7), None, None, None)]:
        u = rng.normal(size=(4, 3)) + 1j * rng.normal(size=(4, 3))
        psi, p = plane_wave(DIMS, n, u)
        a = 1 - 2 * kappa * np.sum(np.cos(p))
        b = 2 * kappa * np.sin(p)
        if a_ref is not None:
            assert abs(a - a_ref) < 1e-9 and abs(np.linalg.norm(b) - b_ref) < 1e-9
        S = a * np.eye(4) + 1j * sum(b[mu] * dbf.GAMMA[mu] for mu in range(4))
        expect = np.einsum("st,...tc->...sc", S, psi)
        got = oracle_lib.M(DIMS, U, A, kappa, psi).reshape(psi.shape)
        assert rel(got, expect) < 1e-14
        ratio = np.linalg.norm(got) ** 2 / np.linalg.norm(psi) ** 2
        assert abs(ratio - (a * a + b @ b)) < 1e-12
        if n2_ref is not None and not np.isnan(n2_ref):
            assert abs(ratio - n2_ref) < 1e-9
        # eigenvalues a +- i|b| (each twice)
        ev = np.sort_complex(np.linalg.eigvals(S))
        assert np.allclose(np.sort(ev.imag), np.sort([-np.linalg.norm(b)] * 2 + [np.linalg.norm(b)] * 2), atol=1e-12)
        assert np.allclose(ev.real, a, atol=1e-12)


def test_periodic_time_boundary_changes_momentum(oracle_lib):
    """t_bc=+1 -> p_t = 2 pi n_t / L_t: the boundary sign is the only thing that moves."""
    kappa = 0.11
    U = inputs.unit_links(DIMS)
    A = oracle_lib.clover(DIMS, U, kappa, 1.0)
    x, y, z, t = lex_coords(DIMS)
    n = (1, 0, 3, 2)
    p = np.array([2 * np.pi * n[k] / DIMS[k] for k in range(4)])
    u = np.arange(12).reshape(4, 3) + 1j
    psi = np.exp(1j * (p[0] * x + p[1] * y + p[2] * z + p[3] * t))[..., None, None] * u
    S = (1 - 2 * kappa * np.sum(np.cos(p))) * np.eye(4) + 2j * kappa * sum(np.sin(p[mu]) * dbf.GAMMA[mu] for mu in range(4))
    got = oracle_lib.M(DIMS, U, A, kappa, psi, t_bc=+1).reshape(psi.shape)
    assert rel(got, np.einsum("st,...tc->...sc", S, psi)) < 1e-14
    bad = oracle_lib.M(DIMS, U, A, kappa, psi, t_bc=-1).reshape(psi.shape)
    assert rel(bad, np.einsum("st,...tc->...sc", S, psi)) > 1e-2


def test_twisted_free_field(oracle_lib):
    """Constant diagonal links U_mu = diag(exp(i theta_mu^c)): colour c sees p_mu + theta_mu^c (pins U vs U^dag
    placement and the colour index order)."""
    kappa = 0.12
    rng = np.random.default_rng(11)
    theta = rng.uniform(-1, 1, size=(4, 3))
    theta[:, 2] = -theta[:, 0] - theta[:, 1]
    U = inputs.unit_links(DIMS)
    for mu in range(4):
        for c in range(3):
            U[mu, ..., c, c] = np.exp(1j * theta[mu, c])
    A = oracle_lib.clover(DIMS, U, kappa, 1.3)
    assert np.abs(A.reshape(-1, 12, 12) - np.eye(12)).max() < 1e-15       # F = 0
    u = rng.normal(size=(4, 3)) + 1j * rng.normal(size=(4, 3))
    psi, p = plane_wave(DIMS, (2, 1, 3, 4), u)
    got = oracle_lib.M(DIMS, U, A, kappa, psi).reshape(psi.shape)
    expect = np.empty_like(psi)
    for c in range(3):
        pc = p + theta[:, c]
        S = (1 - 2 * kappa * np.sum(np.cos(pc))) * np.eye(4) + 2j * kappa * sum(np.sin(pc[mu]) * dbf.GAMMA[mu] for mu in range(4))
        expect[..., c] = np.einsum("st,...t->...s", S, psi[..., c])
    assert rel(got, expect) < 1e-14


# ------------------------------------------------------------------ clover closed form
def uniform_flux_links(dims, nflux):
    Lx, Ly, Lz, Lt = dims
    T = np.array([1.0, -1.0, 0.0])
    B = 2 * np.pi * nflux / (Lx * Ly)
    U = inputs.unit_links(dims)
    x, y, z, t = lex_coords(dims)
    for c in range(3):
        U[0, ..., c, c] = np.exp(-1j * B * y * T[c])
        U[1, ..., c, c] = np.where(y == Ly - 1, np.exp(1j * B * Ly * x * T[c]), 1.0)
    return U, B, T


def test_uniform_flux_clover(oracle_lib):
    """F_xy = sin(B) T at every site, other planes 0, A = 1 - kappa csw sin(B) sigma_xy (x) T
    (pins normalisation 1/8i, leaf orientation, sign and the spin (x) colour index order)."""
    kappa, csw = 0.124, 1.2
    U, B, T = uniform_flux_links(DIMS, 1)
    F = oracle_lib.field_strength(DIMS, U)
    expect = np.zeros_like(F)
    for c in range(3):
        expect[0, ..., c, c] = np.sin(B) * T[c]
    assert np.abs(F - expect).max() < 1e-15
    A = oracle_lib.clover(DIMS, U, kappa, csw)
    sig_xy = np.diag([1.0, -1.0, 1.0, -1.0])
    Aexp = np.eye(12) - kappa * csw * np.sin(B) * np.kron(sig_xy, np.diag(T))
    assert np.abs(A.reshape(-1, 12, 12) - Aexp).max() < 1e-15


def test_uniform_flux_other_plane(oracle_lib):
    """Same field rotated into the z-t plane (directions relabelled): F_zt = sin(B) T, F_xy = 0.
    Catches plane-ordering / sigma_{mu nu} index mistakes the x-y case cannot see."""
    dims = (4, 4, 4, 8)
    Lx, Ly, Lz, Lt = dims
    T = np.array([1.0, -1.0, 0.0])
    B = 2 * np.pi / (Lz * Lt)
    U = inputs.unit_links(dims)
    x, y, z, t = lex_coords(dims)
    for c in range(3):
        U[2, ..., c, c] = np.exp(-1j * B * t * T[c])
        U[3, ..., c, c] = np.where(t == Lt - 1, np.exp(1j * B * Lt * z * T[c]), 1.0)
    F = oracle_lib.field_strength(dims, U)
    expect = np.zeros_like(F)
    for c in range(3):
        expect[5, ..., c, c] = np.sin(B) * T[c]
    assert np.abs(F - expect).max() < 1e-15
    A = oracle_lib.clover(dims, U, 0.12, 1.0)
    sig_zt = 0.5j * (dbf.GAMMA[2] @ dbf.GAMMA[3] - dbf.GAMMA[3] @ dbf.GAMMA[2])
    Aexp = np.eye(12) - 0.12 * np.sin(B) * np.kron(sig_zt, np.diag(T))
    assert np.abs(A.reshape(-1, 12, 12) - Aexp).max() < 1e-15


def test_clover_structure(oracle_lib):
    kappa, csw = 0.12, 1.0
    U = inputs.make_links(DIMS, 1000, 0.3)
    A = oracle_lib.clover(DIMS, U, kappa, csw).reshape(-1, 12, 12)
    assert np.abs(A - A.conj().transpose(0, 2, 1)).max() < 1e-15
    assert np.abs(A[:, :6, 6:]).max() == 0 and np.abs(A[:, 6:, :6]).max() == 0
    assert np.abs(np.trace(A, axis1=1, axis2=2) - 12).max() < 1e-13
    assert np.abs(A - np.eye(12)).max() > 1e-3
    A0 = oracle_lib.clover(DIMS, U, kappa, 0.0).reshape(-1, 12, 12)
    assert np.array_equal(A0, np.broadcast_to(np.eye(12), A0.shape))
    Ainv = oracle_lib.clover_inverse(A)
    assert np.abs(A @ Ainv.reshape(-1, 12, 12) - np.eye(12)).max() < 1e-14
    assert np.abs(Ainv.reshape(-1, 12, 12) - np.linalg.inv(A)).max() < 1e-13
    F = oracle_lib.field_strength(DIMS, U).reshape(6, -1, 3, 3)
    assert np.abs(F - F.conj().transpose(0, 1, 3, 2)).max() < 1e-15          # Hermitian
    assert np.abs(np.trace(F, axis1=2, axis2=3)).max() > 1e-4                # no trace subtraction (reading #5)


# ------------------------------------------------------------------ invariants on arbitrary links
@pytest.fixture(scope="module")
def rough(oracle_lib):
    kappa, csw = 0.12, 1.0
    U = inputs.make_links(DIMS, 1000, 0.3)
    A = oracle_lib.clover(DIMS, U, kappa, csw)
    Ainv = oracle_lib.clover_inverse(A)
    psi = inputs.gaussian_spinors(DIMS, 2, 2000)
    return dict(kappa=kappa, csw=csw, U=U, A=A, Ainv=Ainv, x=psi[0], y=psi[1])


def test_gamma5_hermiticity(oracle_lib, rough):
    r = rough
    My = oracle_lib.M(DIMS, r["U"], r["A"], r["kappa"], r["y"])
    Mdx = oracle_lib.M(DIMS, r["U"], r["A"], r["kappa"], r["x"], dagger=True)
    lhs, rhs = vdot(r["x"], My), vdot(Mdx, r["y"])
    assert abs(lhs - rhs) / abs(lhs) < 1e-14
    # and the dagger really is gamma5 M gamma5 with gamma5 = diag(1,1,-1,-1)
    g5 = np.array([1, 1, -1, -1])[:, None]
    alt = g5 * oracle_lib.M(DIMS, r["U"], r["A"], r["kappa"], g5 * r["x"]).reshape(r["x"].shape)
    assert rel(Mdx.reshape(alt.shape), alt) < 1e-15


def test_hop_anticommutes_with_site_parity(oracle_lib, rough):
    x, y, z, t = lex_coords(DIMS)
    sig = ((-1.0) ** (x + y + z + t))[..., None, None]
    D1 = oracle_lib.hop(DIMS, rough["U"], sig * rough["x"]).reshape(rough["x"].shape)
    D2 = oracle_lib.hop(DIMS, rough["U"], rough["x"]).reshape(rough["x"].shape)
    assert rel(sig * D1, -D2) < 1e-15


def gauge_transform(dims, U, g):
    Ug = np.empty_like(U)
    for mu in range(4):
        gshift = np.roll(g, -1, axis=3 - mu)          # g(x + mu): axes are (t,z,y,x,...)
        Ug[mu] = g @ U[mu] @ gshift.conj().swapaxes(-1, -2)
    return Ug


def test_gauge_covariance(oracle_lib, rough):
    r = rough
    g = inputs.random_gauge_transform(DIMS, 77)
    Ug = gauge_transform(DIMS, r["U"], g)
    Ag = oracle_lib.clover(DIMS, Ug, r["kappa"], r["csw"])
    gpsi = np.einsum("...ab,...sb->...sa", g, r["x"])
    lhs = oracle_lib.M(DIMS, Ug, Ag, r["kappa"], gpsi).reshape(r["x"].shape)
    Mpsi = oracle_lib.M(DIMS, r["U"], r["A"], r["kappa"], r["x"]).reshape(r["x"].shape)
    rhs = np.einsum("...ab,...sb->...sa", g, Mpsi)
    assert rel(lhs, rhs) < 1e-14
    assert rel(lhs, Mpsi) > 0.1      # the transform is not trivial


def test_schur_identity(oracle_lib, rough):
    r = rough
    x, y, z, t = lex_coords(DIMS)
    even = (((x + y + z + t) & 1) == 0)[..., None, None]
    xe = r["x"] * even
    Dx = oracle_lib.hop(DIMS, r["U"], xe).reshape(xe.shape) * (~even)
    xo = r["kappa"] * oracle_lib.apply_site_matrix(r["Ainv"], Dx).reshape(xe.shape)
    full = oracle_lib.M(DIMS, r["U"], r["A"], r["kappa"], xe + xo).reshape(xe.shape)
    mh = oracle_lib.Mhat(DIMS, r["U"], r["A"], r["Ainv"], r["kappa"], r["x"]).reshape(xe.shape)
    assert np.abs(full * (~even)).max() < 1e-14
    assert rel(full * even, mh) < 1e-14
    assert np.abs(mh * (~even)).max() == 0
    # Mhat^dag is the true adjoint of Mhat
    ye = r["y"] * even
    mdy = oracle_lib.Mhat(DIMS, r["U"], r["A"], r["Ainv"], r["kappa"], ye, dagger=True)
    assert abs(vdot(ye, mh) - vdot(mdy, xe)) / abs(vdot(ye, mh)) < 1e-14


# ------------------------------------------------------------------ dense brute force on 2^4
@pytest.fixture(scope="module")
def tiny(oracle_lib):
    dims = (2, 2, 2, 2)
    kappa, csw = 0.12, 1.0
    U = inputs.make_links(dims, 1000, 0.3)
    Md = dbf.dense_M(dims, U, kappa, csw)
    A = oracle_lib.clover(dims, U, kappa, csw)
    return dict(dims=dims, kappa=kappa, csw=csw, U=U, Md=Md, A=A, Ainv=oracle_lib.clover_inverse(A))


def test_dense_2to4_operator(oracle_lib, tiny):
    d = tiny
    assert d["Md"].shape == (192, 192)
    v = inputs.gaussian_spinors(d["dims"], 1, 2000)[0]
    assert rel(oracle_lib.M(d["dims"], d["U"], d["A"], d["kappa"], v).ravel(), d["Md"] @ v.ravel()) < 1e-14
    assert rel(oracle_lib.M(d["dims"], d["U"], d["A"], d["kappa"], v, dagger=True).ravel(), d["Md"].conj().T @ v.ravel()) < 1e-14
    G5 = np.kron(np.eye(16), np.kron(dbf.GAMMA5, np.eye(3)))
    assert np.abs(d["Md"].conj().T - G5 @ d["Md"] @ G5).max() < 1e-14
    Ad = dbf.dense_clover(d["dims"], d["U"], d["kappa"], d["csw"])
    for i in range(16):
        assert np.abs(Ad[12 * i:12 * i + 12, 12 * i:12 * i + 12] - d["A"].reshape(16, 12, 12)[i]).max() < 1e-15
    Dd = dbf.dense_hop(d["dims"], d["U"])
    assert rel(oracle_lib.hop(d["dims"], d["U"], v).ravel(), Dd @ v.ravel()) < 1e-14


def test_dense_2to4_schur_and_solve(oracle_lib, tiny):
    d = tiny
    b = inputs.gaussian_spinors(d["dims"], 1, 2001)[0]
    par = np.repeat(dbf.parity_vector(d["dims"]), 12)
    e, o = par == 0, par == 1
    Md = d["Md"]
    Mhat_dense = Md[np.ix_(e, e)] - Md[np.ix_(e, o)] @ np.linalg.solve(Md[np.ix_(o, o)], Md[np.ix_(o, e)])
    got = oracle_lib.Mhat(d["dims"], d["U"], d["A"], d["Ainv"], d["kappa"], b).ravel()
    assert rel(got[e], Mhat_dense @ b.ravel()[e]) < 1e-14
    bhat = oracle_lib.schur_source(d["dims"], d["U"], d["Ainv"], d["kappa"], b).ravel()
    bhat_dense = b.ravel()[e] - Md[np.ix_(e, o)] @ np.linalg.solve(Md[np.ix_(o, o)], b.ravel()[o])
    assert rel(bhat[e], bhat_dense) < 1e-14
    xd = np.linalg.solve(Md, b.ravel())
    x1, it1, r1 = oracle_lib.solve_eo(d["dims"], d["U"], d["A"], d["Ainv"], d["kappa"], b, 1e-12)
    x2, it2, r2 = oracle_lib.solve_full(d["dims"], d["U"], d["A"], d["kappa"], b, 1e-12)
    assert it1 > 0 and it2 > 0 and r1 <= 1e-12 and r2 <= 1e-12
    assert rel(x1.ravel(), xd) < 1e-11 and rel(x2.ravel(), xd) < 1e-11
    assert np.linalg.cond(Md) < 50


# ------------------------------------------------------------------ solver on configs[0]
def test_config0_solve(oracle_lib, rough):
    r = rough
    b = inputs.gaussian_spinors(DIMS, 1, 2000)[0]
    x, it, res = oracle_lib.solve_eo(DIMS, r["U"], r["A"], r["Ainv"], r["kappa"], b, 1e-10)
    assert 0 < it < 200 and res <= 1e-10
    true_res = np.linalg.norm(b.ravel() - oracle_lib.M(DIMS, r["U"], r["A"], r["kappa"], x).ravel()) / np.linalg.norm(b.ravel())
    assert true_res <= 1.0000001e-10 and abs(true_res - res) < 1e-13
    x2, it2, res2 = oracle_lib.solve_full(DIMS, r["U"], r["A"], r["kappa"], b, 1e-10)
    assert it2 > 0 and rel(x, x2) < 1e-9
    assert it <= it2           # even-odd preconditioning does not make CG slower


# ------------------------------------------------------------------ site-local evaluator
def _all_sites(dims, parity):
    x, y, z, t = lex_coords(dims)
    m = ((x + y + z + t) % 2 == parity)
    return np.stack([x[m], y[m], z[m], t[m]], axis=1).astype(np.int32)


def test_site_local_evaluator_matches_full_lattice(oracle_lib):
    """The per-site routine used for full-size parity (32^3x64, 64^3x128) against the pinned full-lattice
    operator on host arrays: hop, kernel A = A^-1 D, kernel B = A x - kappa^2 D y, every odd / even site."""
    import oracle
    dims, kappa, csw = (4, 6, 4, 8), 0.124, 1.1
    U = inputs.make_links(dims, 31, 0.3)
    psi = inputs.gaussian_spinors(dims, 1, 32)[0].reshape(-1, 12)
    xin = inputs.gaussian_spinors(dims, 1, 33)[0].reshape(-1, 12)
    A = oracle.clover(dims, U, kappa, csw)
    Ainv = oracle.clover_inverse(A)
    Lx, Ly, Lz, Lt = dims
    full_hop = oracle.hop(dims, U, psi).reshape(Lt, Lz, Ly, Lx, 4, 3)
    full_A = oracle.apply_site_matrix(Ainv, full_hop.reshape(-1, 12)).reshape(Lt, Lz, Ly, Lx, 4, 3)
    full_B = (oracle.apply_site_matrix(A, xin) - kappa ** 2 * full_hop.reshape(-1, 12)).reshape(Lt, Lz, Ly, Lx, 4, 3)
    for parity in (0, 1):
        s = _all_sites(dims, parity)
        pick = lambda f: f[s[:, 3], s[:, 2], s[:, 1], s[:, 0]]
        assert rel(oracle.site_eval(dims, 0, s, kappa, csw, U=U, psi=psi), pick(full_hop)) < 1e-14
        assert rel(oracle.site_eval(dims, 1, s, kappa, csw, U=U, psi=psi), pick(full_A)) < 1e-13
        assert rel(oracle.site_eval(dims, 2, s, kappa, csw, coef=-kappa ** 2, U=U, psi=psi, xin=xin), pick(full_B)) < 1e-14


def test_site_local_generator_matches_input_recipe(oracle_lib):
    """The oracle's own C copy of the counter-based generator (links, spinors of any RHS index) against the numpy
    statement of the recipe in inputs.py: regenerated inputs give the same outputs as host arrays."""
    import oracle
    dims, kappa, csw, eps = (4, 4, 6, 4), 0.12, 1.0, 0.3
    U = inputs.make_links(dims, 1002, eps)
    psi = inputs.gaussian_spinors(dims, 3, 7001)
    xin = inputs.gaussian_spinors(dims, 3, 7002)
    s = _all_sites(dims, 1)
    for k in (0, 2):
        want = oracle.site_eval(dims, 2, s, kappa, csw, coef=-0.3, U=U, psi=psi[k].reshape(-1, 12), xin=xin[k].reshape(-1, 12))
        got = oracle.site_eval(dims, 2, s, kappa, csw, coef=-0.3, rhs=k, gauge_seed=1002, eps=eps, in_seed=7001, x_seed=7002)
        assert rel(got, want) < 1e-13
    # periodic time boundary flag is honoured by the site routine too
    a = oracle.site_eval(dims, 0, s, kappa, csw, t_bc=+1, U=U, psi=psi[0].reshape(-1, 12))
    b = oracle.hop(dims, U, psi[0].reshape(-1, 12), t_bc=+1).reshape(dims[3], dims[2], dims[1], dims[0], 4, 3)[s[:, 3], s[:, 2], s[:, 1], s[:, 0]]
    assert rel(a, b) < 1e-14


# ------------------------------------------------------------------ 3-d covariant Laplacian
def _colour_fields(dims, nvec, seed):
    Lx, Ly, Lz, Lt = dims
    idx = np.arange(nvec * Lt * Lz * Ly * Lx * 3, dtype=np.int64)
    return inputs.cgauss(seed, inputs.STREAM_COLORVEC, idx).reshape(nvec, Lt, Lz, Ly, Lx, 3)


def test_laplacian_free_field_closed_form(oracle_lib):
    """U = 1: plane waves exp(i p.x) f(t) chi are eigenvectors with eigenvalue -sum_i 4 sin^2(p_i/2), for ANY time profile
    f(t) (time-slices are independent) and any colour vector chi."""
    import oracle
    dims = (4, 6, 4, 4)
    U = inputs.unit_links(dims)
    x, y, z, t = lex_coords(dims)
    for n in [(1, 2, 3), (0, 0, 0), (3, 5, 1)]:
        p = [2 * np.pi * n[i] / dims[i] for i in range(3)]
        lam = -sum(4 * np.sin(pi / 2) ** 2 for pi in p)
        f = np.exp(1.3j * t) * (1 + t)                      # arbitrary time dependence
        chi = np.array([0.3 - 1j, 2.0, -0.5j])
        v = (np.exp(1j * (p[0] * x + p[1] * y + p[2] * z)) * f)[..., None] * chi
        out = oracle.laplacian(dims, U, v[None])[0]
        assert np.abs(out - lam * v).max() < 1e-12


def test_laplacian_twisted_links_place_U_and_Udag(oracle_lib):
    """Constant diagonal links U_i = diag(exp(i theta_i^c)): colour c sees p_i -> p_i + theta_i^c.  A swapped U / U^dag or a
    transposed colour index changes the eigenvalue."""
    import oracle
    dims = (4, 4, 6, 2)
    rng = np.random.default_rng(3)
    theta = rng.uniform(-1, 1, (3, 3)); theta[:, 2] = -theta[:, 0] - theta[:, 1]
    U = inputs.unit_links(dims).copy()
    for mu in range(3):
        U[mu] = np.diag(np.exp(1j * theta[mu]))
    x, y, z, t = lex_coords(dims)
    n = (1, 3, 2)
    p = [2 * np.pi * n[i] / dims[i] for i in range(3)]
    for c in range(3):
        chi = np.zeros(3, complex); chi[c] = 1.0
        v = np.exp(1j * (p[0] * x + p[1] * y + p[2] * z))[..., None] * chi
        lam = -sum(4 * np.sin((p[i] + theta[i, c]) / 2) ** 2 for i in range(3))
        out = oracle.laplacian(dims, U, v[None])[0]
        assert np.abs(out - lam * v).max() < 1e-12


def test_laplacian_hermitian_negative_covariant_and_time_local(oracle_lib, rough):
    import oracle
    dims, U = DIMS, rough["U"]
    u, v = _colour_fields(dims, 2, 41)
    Lu, Lv = oracle.laplacian(dims, U, np.stack([u, v]))
    assert abs(vdot(u, Lv) - vdot(Lu, v)) < 1e-10 * abs(vdot(u, Lv))          # Hermitian
    assert vdot(v, Lv).real < 0 and abs(vdot(v, Lv).imag) < 1e-10             # negative (semi-)definite
    g = inputs.random_gauge_transform(dims, 42)                                # g[t][z][y][x][3][3]
    Ug = np.empty_like(U)
    for mu in range(4):
        gs = np.roll(g, -1, axis=3 - mu)                                       # g(x + mu)
        Ug[mu] = g @ U[mu] @ np.conj(np.swapaxes(gs, -1, -2))
    gv = np.einsum("...ab,...b->...a", g, v)
    lhs = oracle.laplacian(dims, Ug, gv[None])[0]
    assert rel(lhs, np.einsum("...ab,...b->...a", g, Lv)) < 1e-13              # Lap[U^g](g v) = g Lap[U] v
    # time-slices do not talk to each other, and the time links are never read
    w = v.copy(); w[1:] = 0
    U2 = U.copy(); U2[3] = inputs.make_links(dims, 99, 0.3)[3]
    assert np.abs(oracle.laplacian(dims, U2, w[None])[0][1:]).max() == 0
    assert np.array_equal(oracle.laplacian(dims, U2, w[None])[0][0], Lv[0])


def test_laph_eigen_free_field_and_gauge_invariance(oracle_lib):
    """Dense eigen-decomposition of -Laplacian per time-slice: free-field spectrum = the multiset {sum_i 4 sin^2(p_i/2)} x 3
    colours; the spectrum on rough links is invariant under a gauge transformation; A v = lambda v holds for what comes back."""
    import oracle
    dims = (4, 4, 2, 2)
    ev, vec = oracle.laph_eigen(dims, inputs.unit_links(dims), 12)
    ps = sorted(sum(4 * np.sin(np.pi * n[i] / dims[i]) ** 2 for i in range(3)) for n in np.ndindex(4, 4, 2) for _ in range(3))
    assert np.allclose(ev[0], ps[:12], atol=1e-12) and np.allclose(ev[1], ps[:12], atol=1e-12)
    U = inputs.make_links(dims, 17, 0.3)
    ev, vec = oracle.laph_eigen(dims, U, 10)
    g = inputs.random_gauge_transform(dims, 18)
    Ug = np.empty_like(U)
    for mu in range(4):
        Ug[mu] = g @ U[mu] @ np.conj(np.swapaxes(np.roll(g, -1, axis=3 - mu), -1, -2))
    ev_g, _ = oracle.laph_eigen(dims, Ug, 10)
    assert np.allclose(ev, ev_g, atol=1e-12)
    assert np.all(ev > -1e-12) and np.all(np.diff(ev, axis=1) >= -1e-12)
    v = np.zeros((10, 2, 2, 4, 4, 3), dtype=complex)
    v[:, 1] = vec[1]                                   # the slice-1 eigenvectors, zero elsewhere
    Lv = oracle.laplacian(dims, U, v)
    assert np.abs(-Lv[:, 1] - ev[1][:, None, None, None, None] * v[:, 1]).max() < 1e-12


def test_projection_definition_and_invariants(oracle_lib):
    """P[t][a][j][k] = <v_j(t), psi_k(t, a)>: explicit loops on a tiny case, recovery of expansion coefficients in an
    orthonormal basis, gauge invariance."""
    import oracle
    dims = (2, 2, 2, 3)
    Lx, Ly, Lz, Lt = dims
    rng = np.random.default_rng(8)
    v = rng.normal(size=(3, Lt, Lz, Ly, Lx, 3)) + 1j * rng.normal(size=(3, Lt, Lz, Ly, Lx, 3))
    psi = rng.normal(size=(2, Lt, Lz, Ly, Lx, 4, 3)) + 1j * rng.normal(size=(2, Lt, Lz, Ly, Lx, 4, 3))
    P = oracle.project(v, psi)
    for t in range(Lt):
        for a in range(4):
            for j in range(3):
                for k in range(2):
                    s = 0
                    for z in range(Lz):
                        for y in range(Ly):
                            for x in range(Lx):
                                for c in range(3):
                                    s += np.conj(v[j, t, z, y, x, c]) * psi[k, t, z, y, x, a, c]
                    assert abs(P[t, a, j, k] - s) < 1e-12
    # orthonormal basis per slice (QR) and a field inside its span: the projection returns the coefficients
    q = np.empty_like(v)
    for t in range(Lt):
        Q, _ = np.linalg.qr(v[:, t].reshape(3, -1).T)
        q[:, t] = Q.T.reshape(3, Lz, Ly, Lx, 3)
    coef = rng.normal(size=(Lt, 4, 3, 2)) + 1j * rng.normal(size=(Lt, 4, 3, 2))
    field = np.einsum("tajk,jtzyxc->ktzyxac", coef, q)
    assert np.abs(oracle.project(q, field) - coef).max() < 1e-12
    # gauge invariance
    g = inputs.random_gauge_transform(dims, 9)
    gv = np.einsum("tzyxab,jtzyxb->jtzyxa", g, v)
    gpsi = np.einsum("tzyxab,ktzyxsb->ktzyxsa", g, psi)
    assert np.abs(oracle.project(gv, gpsi) - P).max() < 1e-11


def test_int16_link_quantisation_error_of_the_operator(oracle_lib):
    """SURVEY 8(c.2) reading #13 (the oracle-side check of the int16-link solver variant): quantising every link entry to
    q = rint(32767 u) / 32767 changes M psi by a few 1e-5 relative (survey scratch: 3.5e-5), far below the half-storage tolerance."""
    dims = (4, 4, 4, 8)
    U = inputs.make_links(dims, 1000, 0.3)
    Uq = (np.rint(U.view(np.float64) * 32767.0) / 32767.0).view(np.complex128)
    oracle = oracle_lib
    A = oracle.clover(dims, U, 0.12, 1.0)
    psi = inputs.gaussian_spinors(dims, 1, 2000)[0]
    ref = oracle.M(dims, U, A, 0.12, psi)
    err = np.linalg.norm(oracle.M(dims, Uq, A, 0.12, psi) - ref) / np.linalg.norm(ref)
    assert 1e-7 < err < 1e-4, err
