"""GPU parity of the time-batched Lanczos eigensolver against the oracle's dense per-slice
eigen-decomposition: eigenvalues, residuals, orthonormality per slice, and the spanned subspace."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle  # noqa: E402
from paper_2510_26313_b200 import binding as B, inputs  # noqa: E402


@pytest.mark.parametrize("dims,n_ev,m,deg", [((4, 4, 4, 4), 8, 24, 6), ((6, 4, 4, 2), 5, 16, 8), ((4, 4, 2, 6), 12, 30, 5),
                                              ((4, 4, 4, 2), 70, 110, 6)])          # Krylov space beyond 64: tiled rotation, threaded Ritz step
def test_lanczos_matches_dense_eigh(dims, n_ev, m, deg):
    U = inputs.make_links(dims, 71, 0.3)
    Lx, Ly, Lz, Lt = dims
    ev_o, vec_o = oracle.laph_eigen(dims, U, n_ev + 4)
    ctx = B.Context(dims)
    ctx.load_gauge(U)
    cut = 0.5 * (ev_o[:, n_ev + 1].max() + ev_o[:, n_ev + 3].max())          # just above the wanted part of every slice
    ev, vec, info = ctx.laph_eigensolve(n_ev, m, deg, cheb_a=cut, cheb_b=12.5, tol=1e-11, max_restarts=200)
    ctx.close()
    assert info["converged"], info
    assert np.abs(ev - ev_o[:, :n_ev]).max() <= 1e-9, (np.abs(ev - ev_o[:, :n_ev]).max(), info)
    assert info["max_true_residual"] <= 1e-7
    # the returned vectors: unit norm and mutually orthogonal on every slice, A v = lambda v by the ORACLE's operator
    Lv = oracle.laplacian(dims, U, vec)
    for t in range(Lt):
        Vt = vec[:, t].reshape(n_ev, -1)
        assert np.abs(Vt.conj() @ Vt.T - np.eye(n_ev)).max() <= 1e-9
        R = -Lv[:, t].reshape(n_ev, -1) - ev[t][:, None] * Vt
        assert np.abs(R).max() <= 1e-7
        # same subspace as the dense solver for the part of the spectrum separated by a gap
        gaps = np.diff(ev_o[t, :n_ev + 1])
        j = int(np.argmax(gaps[n_ev // 2:])) + n_ev // 2 + 1                  # cluster = the lowest j states
        Po = vec_o[t, :j].reshape(j, -1)
        sv = np.linalg.svd(Po.conj() @ Vt[:j].T, compute_uv=False)
        assert sv.min() >= 1 - 1e-6


def test_eigensolve_reports_non_convergence_and_bad_parameters():
    dims = (4, 4, 4, 2)
    ctx = B.Context(dims)
    ctx.load_gauge(inputs.make_links(dims, 72, 0.3))
    ev, vec, info = ctx.laph_eigensolve(6, 12, 2, cheb_a=3.0, tol=1e-14, max_restarts=1)
    assert not info["converged"] and ev.shape == (2, 6)
    with pytest.raises(B.LqError):
        ctx.laph_eigensolve(6, 7, 4, cheb_a=1.0)           # m < n_ev + 2
    with pytest.raises(B.LqError):
        ctx.laph_eigensolve(6, 16, 4, cheb_a=13.0)         # cut above the upper bound
    ctx.close()
