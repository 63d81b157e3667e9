"""GPU parity of the eigenvector projection against the oracle's einsum, and the LapH chain
eigensolve -> solve -> project on one small lattice."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle  # noqa: E402
from paper_2510_26313_b200 import binding as B, inputs  # noqa: E402


@pytest.mark.parametrize("dims,n_ev,n_sol", [((4, 4, 4, 4), 5, 3), ((6, 4, 2, 6), 8, 4), ((8, 8, 8, 2), 13, 1), ((2, 2, 2, 2), 1, 2)])
def test_projection_matches_einsum(dims, n_ev, n_sol):
    Lx, Ly, Lz, Lt = dims
    rng = np.random.default_rng(5)
    v = rng.normal(size=(n_ev, Lt, Lz, Ly, Lx, 3)) + 1j * rng.normal(size=(n_ev, Lt, Lz, Ly, Lx, 3))
    psi = inputs.gaussian_spinors(dims, n_sol, 81)
    want = oracle.project(v, psi)
    ctx = B.Context(dims)
    got = ctx.project(v, psi)
    got_tc = ctx.project(v, psi, B.LQ_FP32)          # tcgen05 tensor cores, 3xTF32
    ctx.close()
    assert np.abs(got - want).max() <= 1e-12 * np.abs(want).max() * np.sqrt(3 * Lx * Ly * Lz)
    assert np.abs(got_tc - want).max() <= 3e-6 * np.abs(want).max()


def test_tensor_core_projection_tiles_and_padding():
    """More eigenvectors than one 128-row tile, more solutions than one 8-solution tile, a slice that is not a multiple of the
    256-site K chunk or the 16-site block."""
    dims, n_ev, n_sol = (6, 6, 10, 2), 150, 11
    Lx, Ly, Lz, Lt = dims
    rng = np.random.default_rng(6)
    v = rng.normal(size=(n_ev, Lt, Lz, Ly, Lx, 3)) + 1j * rng.normal(size=(n_ev, Lt, Lz, Ly, Lx, 3))
    psi = inputs.gaussian_spinors(dims, n_sol, 82)
    want = oracle.project(v, psi)
    ctx = B.Context(dims)
    got_tc = ctx.project(v, psi, B.LQ_FP32)
    ctx.close()
    assert np.abs(got_tc - want).max() <= 3e-6 * np.abs(want).max()


def test_projection_is_bitwise_reproducible():
    """Both kernels sum in a fixed order (no atomics): two calls on the same inputs return identical bits."""
    import torch
    dims, n_ev, n_sol = (8, 8, 8, 4), 40, 12
    Lx, Ly, Lz, Lt = dims
    g = torch.Generator(device="cuda").manual_seed(3)
    v = torch.view_as_complex(torch.randn((n_ev, Lt, Lz, Ly, Lx, 3, 2), generator=g, device="cuda", dtype=torch.float64))
    x = torch.view_as_complex(torch.randn((n_sol, Lt, Lz, Ly, Lx, 4, 3, 2), generator=g, device="cuda", dtype=torch.float64))
    ctx = B.Context(dims)
    for prec in (B.LQ_FP64, B.LQ_FP32):
        a = ctx.project(v, x, prec)
        b = ctx.project(v, x, prec)
        assert torch.equal(torch.view_as_real(a), torch.view_as_real(b))
    ctx.close()


def test_projection_bench_size_sampled():
    """The shape bench.py times (16^3x32, 128 eigenvectors x 32 solutions, device arrays): sampled outputs against the oracle's
    einsum on the matching slices, and the tensor-core kernel against the fp64 kernel on every output."""
    import torch
    dims, n_ev, n_sol = inputs.CONFIGS[1]["dims"], 128, 32
    Lx, Ly, Lz, Lt = dims
    g = torch.Generator(device="cuda").manual_seed(7)
    v = torch.view_as_complex(torch.randn((n_ev, Lt, Lz, Ly, Lx, 3, 2), generator=g, device="cuda", dtype=torch.float64))
    x = torch.view_as_complex(torch.randn((n_sol, Lt, Lz, Ly, Lx, 4, 3, 2), generator=g, device="cuda", dtype=torch.float64))
    ctx = B.Context(dims)
    p64 = ctx.project(v, x)
    ptc = ctx.project(v, x, B.LQ_FP32)
    ctx.close()
    scale = p64.abs().max().item()
    assert (ptc - p64).abs().max().item() <= 3e-6 * scale
    rng = np.random.default_rng(11)
    for _ in range(24):
        t, j, k = int(rng.integers(Lt)), int(rng.integers(n_ev)), int(rng.integers(n_sol))
        want = oracle.project(v[j:j + 1, t:t + 1].cpu().numpy(), x[k:k + 1, t:t + 1].cpu().numpy())     # [1][4][1][1]
        got64 = p64[t, :, j, k].cpu().numpy()
        gottc = ptc[t, :, j, k].cpu().numpy()
        assert np.abs(got64 - want[0, :, 0, 0]).max() <= 1e-12 * scale
        assert np.abs(gottc - want[0, :, 0, 0]).max() <= 3e-6 * scale


def test_laph_chain_eigensolve_solve_project():
    """Sources built from GPU eigenvectors of one time-slice, propagated by lq_solve, projected back: compared with the same
    chain done by the oracle (dense eigenvectors fix the phases, so the GPU vectors are used for both projections)."""
    dims, kappa, csw = (4, 4, 4, 8), 0.12, 1.0
    U = inputs.make_links(dims, 91, 0.3)
    ctx = B.Context(dims)
    ctx.load_gauge(U)
    ctx.build_clover(kappa, csw)
    ev, vec, info = ctx.laph_eigensolve(4, 16, 6, cheb_a=2.0, tol=1e-11)
    assert info["converged"]
    b = np.zeros((4, dims[3], dims[2], dims[1], dims[0], 4, 3), dtype=np.complex128)
    for k in range(4):
        b[k, 0, :, :, :, k % 4, :] = vec[0, 0]            # LapH source: eigenvector 0 on time-slice 0, spin k
    x, sinfo = ctx.solve(b, tol=1e-10, inner_prec=B.LQ_FP32, delta=1e-3)
    assert sinfo["converged"]
    P = ctx.project(vec, x)
    ctx.close()
    A = oracle.clover(dims, U, kappa, csw); Ainv = oracle.clover_inverse(A)
    xo = np.stack([oracle.solve_eo(dims, U, A, Ainv, kappa, b[k], 1e-12)[0].reshape(b[k].shape) for k in range(4)])
    Po = oracle.project(vec, xo)
    assert np.abs(P - Po).max() <= 1e-8 * np.abs(Po).max()


@pytest.mark.parametrize("dims,n_ev,n_sol", [((4, 4, 4, 4), 5, 3), ((6, 4, 2, 6), 8, 4), ((8, 8, 8, 2), 13, 1), ((2, 2, 2, 2), 1, 2), ((6, 6, 10, 2), 150, 11)])
def test_single_precision_fields_match_einsum(dims, n_ev, n_sol):
    """lq_project_c64: complex64 fields in, the oracle's einsum on exactly those (rounded) fields as the reference; tiles, padding,
    ragged K chunks and both kernel shapes (n_sol <= 8: N = 64 with 8-site stages; more: N = 256 with 4-site stages)."""
    Lx, Ly, Lz, Lt = dims
    rng = np.random.default_rng(15)
    v = (rng.normal(size=(n_ev, Lt, Lz, Ly, Lx, 3)) + 1j * rng.normal(size=(n_ev, Lt, Lz, Ly, Lx, 3))).astype(np.complex64)
    psi = inputs.gaussian_spinors(dims, n_sol, 83).astype(np.complex64)
    want = oracle.project(v.astype(np.complex128), psi.astype(np.complex128))
    ctx = B.Context(dims)
    got = ctx.project_c64(v, psi)
    again = ctx.project_c64(v, psi)
    ctx.close()
    assert np.abs(got - want).max() <= 3e-6 * np.abs(want).max()
    assert np.array_equal(got, again)                     # fixed summation order


def test_single_precision_projection_bench_size():
    """16^3 x 32, 128 x 32, device arrays: every output against the fp64 FMA kernel run on the same (rounded) fields."""
    import torch
    dims, n_ev, n_sol = inputs.CONFIGS[1]["dims"], 128, 32
    Lx, Ly, Lz, Lt = dims
    g = torch.Generator(device="cuda").manual_seed(9)
    v = torch.view_as_complex(torch.randn((n_ev, Lt, Lz, Ly, Lx, 3, 2), generator=g, device="cuda", dtype=torch.float32))
    x = torch.view_as_complex(torch.randn((n_sol, Lt, Lz, Ly, Lx, 4, 3, 2), generator=g, device="cuda", dtype=torch.float32))
    ctx = B.Context(dims)
    p32 = ctx.project_c64(v, x)
    p64 = ctx.project(v.to(torch.complex128), x.to(torch.complex128))
    ctx.close()
    assert ((p32 - p64).abs().max() / p64.abs().max()).item() <= 3e-6
