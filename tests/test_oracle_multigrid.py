"""Pins of the two-level multigrid oracle (oracle/multigrid.py, PAPER.md L118 / L164), CPU only.

What the mathematics fixes, independent of the code under test: the prolongator has orthonormal columns and reproduces the
near-null vectors it was built from; gamma5 P = P Gamma5_c with Gamma5_c = +-1 on the two chiralities, hence the Galerkin operator
is Gamma5_c-Hermitian like M is gamma5-Hermitian; aggregates couple to nearest neighbours only; the coarse-grid correction is exact
on the range of P; a preconditioned flexible Krylov solve still reaches the solution of M x = b (residual by the pinned oracle.M)
and needs fewer iterations than the unpreconditioned one."""
import numpy as np
import pytest

from paper_2510_26313_b200 import inputs

DIMS, BLOCK, NV = (4, 4, 4, 8), (2, 2, 2, 2), 4
KAPPA, CSW, EPS = 0.128, 1.0, 0.15


@pytest.fixture(scope="module")
def setup(oracle_lib):
    oracle = oracle_lib
    from oracle import multigrid as mg
    U = inputs.make_links(DIMS, 1000, EPS)
    A = oracle.clover(DIMS, U, KAPPA, CSW)
    Ainv = oracle.clover_inverse(A)
    V = inputs.volume(DIMS)

    def apply_M(v):
        return oracle.M(DIMS, U, A, KAPPA, v.reshape(V, 12)).reshape(-1)
    eta = inputs.gaussian_spinors(DIMS, NV, 77)
    vecs = np.stack([oracle.solve_eo(DIMS, U, A, Ainv, KAPPA, eta[k], 1e-3)[0].reshape(eta[k].shape) for k in range(NV)])
    P, Lc = mg.prolongator(DIMS, BLOCK, vecs)
    Ac = mg.coarse_operator(apply_M, P)
    return dict(oracle=oracle, mg=mg, U=U, A=A, Ainv=Ainv, apply_M=apply_M, vecs=vecs, P=P, Lc=Lc, Ac=Ac, V=V)


def test_prolongator_is_orthonormal_and_reproduces_its_vectors(setup):
    P, vecs = setup["P"], setup["vecs"]
    n = P.shape[1]
    assert n == int(np.prod(setup["Lc"])) * 2 * NV
    assert np.allclose(P.conj().T @ P, np.eye(n), atol=1e-12)
    for k in range(NV):
        v = vecs[k].reshape(-1)
        assert np.linalg.norm(P @ (P.conj().T @ v) - v) <= 1e-12 * np.linalg.norm(v)
    # every column lives on one aggregate and one chirality
    a, _ = setup["mg"].aggregate_index(DIMS, BLOCK)
    a = np.repeat(a.reshape(-1), 12)
    chi = np.tile(np.repeat([0, 0, 1, 1], 3), setup["V"])
    for c in range(0, n, 7):
        nz = np.abs(P[:, c]) > 0
        ag, ch = c // (2 * NV), (c // NV) % 2
        assert np.all(a[nz] == ag) and np.all(chi[nz] == ch)


def test_coarse_operator_inherits_gamma5_hermiticity_and_locality(setup):
    Ac, Lc = setup["Ac"], setup["Lc"]
    n = Ac.shape[0]
    g5c = np.tile(np.repeat([1.0, -1.0], NV), n // (2 * NV))
    assert np.allclose(Ac.conj().T, g5c[:, None] * Ac * g5c[None, :], atol=1e-12)
    # blocks between aggregates that are not nearest neighbours (periodic, one direction) vanish
    Vc = n // (2 * NV)
    def coords(a):
        return np.array([a % Lc[0], (a // Lc[0]) % Lc[1], (a // (Lc[0] * Lc[1])) % Lc[2], a // (Lc[0] * Lc[1] * Lc[2])])
    far = near = 0
    for a1 in range(Vc):
        for a2 in range(Vc):
            d = np.abs(coords(a1) - coords(a2))
            d = np.minimum(d, np.array(Lc) - d)
            blk = Ac[a1 * 2 * NV:(a1 + 1) * 2 * NV, a2 * 2 * NV:(a2 + 1) * 2 * NV]
            if d.sum() > 1:
                assert np.all(blk == 0) or np.abs(blk).max() <= 1e-14
                far += 1
            else:
                near += int(np.abs(blk).max() > 1e-8)
    assert far > 0 and near >= Vc


def test_coarse_grid_correction_is_exact_on_the_range_of_P(setup):
    P, Ac, apply_M = setup["P"], setup["Ac"], setup["apply_M"]
    rng = np.random.default_rng(3)
    y = rng.standard_normal(P.shape[1]) + 1j * rng.standard_normal(P.shape[1])
    x = P @ y
    corr = P @ np.linalg.solve(Ac, P.conj().T @ apply_M(x))
    assert np.linalg.norm(x - corr) <= 1e-10 * np.linalg.norm(x)
    # Galerkin condition on an arbitrary coarse vector, with the fine operator applied by the pinned oracle
    assert np.allclose(Ac @ y, P.conj().T @ apply_M(P @ y), atol=1e-11 * np.linalg.norm(y))


def test_two_grid_fgcr_reaches_the_solution_in_fewer_iterations(setup):
    mg, apply_M, P, Ac = setup["mg"], setup["apply_M"], setup["P"], setup["Ac"]
    b = inputs.gaussian_spinors(DIMS, 1, 5)[0].reshape(-1)
    x0, it0, _ = mg.fgcr(apply_M, b, 1e-9, maxit=400, restart=400)          # full GCR: GCR(16) on M stagnates
    x1, it1, hist = mg.fgcr(apply_M, b, 1e-9, precond=lambda r: mg.two_grid_preconditioner(apply_M, P, Ac, r, smooth=2))
    for x in (x0, x1):
        assert np.linalg.norm(b - apply_M(x)) <= 1e-9 * np.linalg.norm(b)
    assert np.linalg.norm(x0 - x1) <= 1e-7 * np.linalg.norm(x0)
    assert it1 < it0 / 2, (it0, it1)
    # reference solution by the oracle's own even-odd CG
    oracle = setup["oracle"]
    xr = oracle.solve_eo(DIMS, setup["U"], setup["A"], setup["Ainv"], KAPPA, b.reshape(-1, 12), 1e-11)[0].reshape(-1)
    assert np.linalg.norm(x1 - xr) <= 1e-7 * np.linalg.norm(xr)


def test_schur_smoother_solves_the_odd_rows_exactly_and_converges_to_the_inverse(setup):
    """LQ_MG_SMOOTH_EO: after any number of steps the odd rows of r - M delta vanish (the reconstruction solves them exactly), the
    even rows shrink monotonically (minimal residual), and many steps approach M^-1 r."""
    mg, oracle, apply_M = setup["mg"], setup["oracle"], setup["apply_M"]
    Lx, Ly, Lz, Lt = DIMS
    t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    odd = np.repeat(((x + y + z + t) & 1).reshape(-1) == 1, 12)
    r = inputs.gaussian_spinors(DIMS, 1, 9)[0].reshape(-1)
    prev = np.inf
    for steps in (0, 1, 3, 6):
        d = mg.schur_mr_smoother(DIMS, setup["U"], setup["A"], setup["Ainv"], KAPPA, r, steps)
        res = r - apply_M(d)
        assert np.linalg.norm(res[odd]) <= 1e-13 * np.linalg.norm(r)
        n = np.linalg.norm(res[~odd])
        assert n < prev
        prev = n
    d = mg.schur_mr_smoother(DIMS, setup["U"], setup["A"], setup["Ainv"], KAPPA, r, 300)
    assert np.linalg.norm(r - apply_M(d)) <= 1e-3 * np.linalg.norm(r)          # MR(1) is slow but it does converge


def test_even_odd_smoother_makes_the_better_cycle(setup):
    mg, apply_M, P, Ac = setup["mg"], setup["apply_M"], setup["P"], setup["Ac"]
    b = inputs.gaussian_spinors(DIMS, 1, 5)[0].reshape(-1)

    def eo(res):
        return mg.schur_mr_smoother(DIMS, setup["U"], setup["A"], setup["Ainv"], KAPPA, res, 2)
    x1, it_mr, _ = mg.fgcr(apply_M, b, 1e-9, precond=lambda r: mg.two_grid_preconditioner(apply_M, P, Ac, r, smooth=2))
    x2, it_eo, _ = mg.fgcr(apply_M, b, 1e-9, precond=lambda r: mg.two_grid_preconditioner(apply_M, P, Ac, r, smoother=eo))
    assert np.linalg.norm(b - apply_M(x2)) <= 1e-9 * np.linalg.norm(b)
    assert np.linalg.norm(x1 - x2) <= 1e-7 * np.linalg.norm(x1)
    assert it_eo < it_mr, (it_eo, it_mr)
