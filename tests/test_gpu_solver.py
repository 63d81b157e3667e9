"""GPU solver parity: true residual recomputed by the oracle's full M, solution vs
the oracle's own CG, every inner precision.  Iteration counts are not compared (parity unpinned, 8(c.3))."""
import numpy as np
import pytest

import oracle
from paper_2510_26313_b200 import inputs
from paper_2510_26313_b200 import binding as B
from tests.oracle_ops import OracleCase, rel_err

pytestmark = pytest.mark.gpu


def true_residuals(orc, x, b):
    out = []
    for k in range(b.shape[0]):
        r = b[k].ravel() - oracle.M(orc.dims, orc.U, orc.A, orc.kappa, x[k], False, orc.t_bc).ravel()
        out.append(np.linalg.norm(r) / np.linalg.norm(b[k].ravel()))
    return np.array(out)


def setup(dims, seed, eps, kappa, csw, recon=18):
    U = inputs.make_links(dims, seed, eps)
    ctx = B.Context(dims)
    ctx.load_gauge(U, recon=recon)
    ctx.build_clover(kappa, csw)
    return ctx, OracleCase(dims, U, kappa, csw)


def test_config0_solve_fp64():
    """configs[0]: 4^3 x 8, 1 RHS, fp64 throughout, even-odd CG on MdagM to 1e-10."""
    cfg = inputs.CONFIGS[0]
    ctx, orc = setup(cfg["dims"], cfg["gauge_seed"], cfg["eps"], cfg["kappa"], cfg["csw"])
    b = inputs.gaussian_spinors(cfg["dims"], 1, cfg["source_seed"])
    x, info = ctx.solve(b, tol=cfg["tol"], inner_prec=B.LQ_FP64, delta=1e-11, check_every=5)
    assert info["converged"]
    res = true_residuals(orc, x, b)
    assert res[0] <= cfg["tol"]
    assert abs(info["true_rel_residual"][0] - res[0]) <= 1e-12          # Schur identity: eo residual = full residual
    xo, it, _ = oracle.solve_eo(cfg["dims"], orc.U, orc.A, orc.Ainv, cfg["kappa"], b[0], cfg["tol"] * 1e-2)
    assert rel_err(x[0], xo.reshape(x[0].shape)) <= 20 * cfg["tol"]     # cond(M) is O(10) on these links
    assert 0 < info["inner_iters"] < 10 * it
    ctx.close()


@pytest.mark.parametrize("inner,delta,tol", [(B.LQ_FP32, 1e-3, 1e-8), (B.LQ_HALF, 1e-2, 1e-9), (B.LQ_FP64, 1e-4, 1e-10)])
@pytest.mark.parametrize("use_graph", [False, True])
def test_batched_mixed_precision_solve(inner, delta, tol, use_graph):
    """8^3 x 16 stand-in for configs[1] / configs[3]: LapH-diluted sources, fp32 / int16 inner CG, fp64 defect correction."""
    dims = (8, 8, 8, 16)
    nrhs = 8 if inner != B.LQ_HALF else 12
    n_t = 2 if inner != B.LQ_HALF else 3
    ctx, orc = setup(dims, 1001, 0.2, 0.124, 1.2)
    b = inputs.laph_sources(dims, nrhs, n_t, 2001)
    x, info = ctx.solve(b, tol=tol, inner_prec=inner, delta=delta, use_graph=use_graph, check_every=4)
    assert info["converged"], info
    res = true_residuals(orc, x, b)
    assert np.all(res <= tol), res
    assert np.allclose(res, info["true_rel_residual"], rtol=1e-3, atol=tol * 1e-3)
    for k in (0, nrhs - 1):
        xo, _, _ = oracle.solve_eo(dims, orc.U, orc.A, orc.Ainv, 0.124, b[k], tol * 1e-2)
        assert rel_err(x[k], xo.reshape(x[k].shape)) <= 50 * tol
    assert info["outer_cycles"] >= 1 and info["inner_iters"] > 0
    ctx.close()


def test_solve_device_buffers_and_native_layout():
    import torch
    dims = (8, 4, 4, 8)
    ctx, orc = setup(dims, 3, 0.3, 0.12, 1.0)
    b = inputs.gaussian_spinors(dims, 4, 9)
    x_host, _ = ctx.solve(b, tol=1e-9, inner_prec=B.LQ_FP32)
    bd = torch.from_numpy(b).cuda()
    xd, info = ctx.solve(bd, tol=1e-9, inner_prec=B.LQ_FP32)
    assert info["converged"] and np.array_equal(xd.cpu().numpy(), x_host)     # deterministic reductions: bit-identical
    nb = ctx.pack(b, 4, B.LQ_FP64)
    nx, info = ctx.solve(nb, tol=1e-9, inner_prec=B.LQ_FP32, native=True, nrhs=4)
    assert np.array_equal(ctx.unpack(nx, 4, B.LQ_FP64), x_host)
    assert np.all(true_residuals(orc, x_host, b) <= 1e-9)
    ctx.close()


def test_zero_and_mixed_difficulty_sources():
    """Degenerate batch: one RHS identically zero, one tiny, one point source; per-RHS alpha/beta guards (reading #18)."""
    dims = (4, 4, 4, 8)
    ctx, orc = setup(dims, 1000, 0.3, 0.12, 1.0)
    b = inputs.gaussian_spinors(dims, 4, 5)
    b[1] = 0
    b[2] *= 1e-12
    b[3] = 0
    b[3, 0, 0, 0, 0, 0, 0] = 1.0
    x, info = ctx.solve(b, tol=1e-9, inner_prec=B.LQ_FP32)
    assert info["converged"] and np.all(np.isfinite(x.view(np.float64)))
    assert np.all(x[1] == 0)
    res = [np.linalg.norm(b[k].ravel() - oracle.M(dims, orc.U, orc.A, 0.12, x[k]).ravel()) / np.linalg.norm(b[k].ravel()) for k in (0, 2, 3)]
    assert max(res) <= 1e-9
    ctx.close()


def test_not_converged_is_reported():
    dims = (4, 4, 4, 8)
    ctx, orc = setup(dims, 1000, 0.3, 0.12, 1.0)
    b = inputs.gaussian_spinors(dims, 2, 5)
    x, info = ctx.solve(b, tol=1e-12, inner_prec=B.LQ_FP32, max_outer=1, max_inner=4, check_every=2)
    assert not info["converged"] and max(info["true_rel_residual"]) > 1e-12
    assert np.all(np.isfinite(x.view(np.float64)))
    ctx.close()


@pytest.mark.parametrize("inner", [B.LQ_FP32, B.LQ_HALF])
def test_solve_is_bitwise_reproducible(inner):
    """The per-RHS reductions (fused kernel-B epilogues and block-BLAS) are fixed-order: two solves of the same system
    give bit-identical solutions and iteration counts, with and without CUDA-graph replay."""
    dims = (8, 8, 8, 8)
    ctx, orc = setup(dims, 77, 0.25, 0.124, 1.1)
    b = inputs.laph_sources(dims, 8, 2, 78)
    runs = []
    for use_graph in (False, False, True):
        x, info = ctx.solve(b, tol=1e-8, inner_prec=inner, delta=1e-2, check_every=4, use_graph=use_graph)
        assert info["converged"]
        runs.append((x.copy(), info["inner_iters"], info["outer_cycles"]))
    for x, it, oc in runs[1:]:
        assert it == runs[0][1] and oc == runs[0][2]
        assert np.array_equal(x, runs[0][0])
    assert np.all(true_residuals(orc, runs[0][0], b) <= 1e-8)
    ctx.close()


@pytest.mark.parametrize("nrhs", [1, 2, 12, 16, 20, 32])
def test_every_batch_width_solves(nrhs):
    """RHS group widths 1, 2 and 4 and 1, 3 and 4 groups per site block through the fused CG iteration (fp32 inner)."""
    dims = (6, 6, 4, 8)          # Vh = 432: 13.5 site blocks, the last one half padding
    ctx, orc = setup(dims, 91, 0.3, 0.123, 1.0)
    b = inputs.gaussian_spinors(dims, nrhs, 92)
    x, info = ctx.solve(b, tol=1e-9, inner_prec=B.LQ_FP32, delta=1e-3, check_every=6, use_graph=True)
    assert info["converged"], info
    assert np.all(true_residuals(orc, x, b) <= 1e-9)
    ctx.close()


@pytest.mark.parametrize("keep_direction", [False, True])
def test_restart_and_reliable_update_variants(keep_direction):
    """Both outer-loop variants (SURVEY 8(c.2) reading #11): restart defect correction (p = z after every fp64 residual
    refresh) and reliable updates (the direction survives the refresh).  Both must reach the tolerance; keeping the
    direction must not cost iterations."""
    dims = (8, 8, 8, 16)
    ctx, orc = setup(dims, 55, 0.25, 0.124, 1.15)
    b = inputs.laph_sources(dims, 8, 2, 56)
    x, info = ctx.solve(b, tol=1e-9, inner_prec=B.LQ_FP32, delta=1e-2, check_every=2, use_graph=True, keep_direction=keep_direction)
    assert info["converged"], info
    assert np.all(true_residuals(orc, x, b) <= 1e-9)
    test_restart_and_reliable_update_variants.iters[keep_direction] = info["inner_iters"]
    if len(test_restart_and_reliable_update_variants.iters) == 2:
        it = test_restart_and_reliable_update_variants.iters
        assert it[True] <= it[False]
    ctx.close()


test_restart_and_reliable_update_variants.iters = {}


def test_config1_full_size_bench_configuration():
    """configs[1] itself (16^3x32, 8 LapH-diluted RHS) in the launch configuration bench.py times (fp32 inner CG, delta 1e-4, poll every
    4 iterations, CUDA-graph replay, reliable updates): the oracle recomputes the true residual of every RHS with its full M, and
    one solution is compared with the oracle's own fp64 CG."""
    cfg = inputs.CONFIGS[1]
    dims, nrhs = cfg["dims"], cfg["nrhs"]
    ctx, orc = setup(dims, cfg["gauge_seed"], cfg["eps"], cfg["kappa"], cfg["csw"])
    b = inputs.laph_sources(dims, nrhs, cfg["n_t"], cfg["source_seed"])
    x, info = ctx.solve(b, tol=cfg["tol"], inner_prec=B.LQ_FP32, delta=1e-4, check_every=4, use_graph=True, keep_direction=True)
    ctx.close()
    assert info["converged"], info
    res = true_residuals(orc, x, b)
    assert np.all(res <= cfg["tol"]), res
    assert np.allclose(res, info["true_rel_residual"], rtol=1e-3, atol=cfg["tol"] * 1e-3)
    k = 5
    xo, _, _ = oracle.solve_eo(dims, orc.U, orc.A, orc.Ainv, cfg["kappa"], b[k], cfg["tol"] * 1e-2)
    assert rel_err(x[k], xo.reshape(x[k].shape)) <= 50 * cfg["tol"]


@pytest.mark.parametrize("inner,delta,tol,nrhs", [(B.LQ_FP32, 1e-3, 1e-8, 8), (B.LQ_FP64, 1e-4, 1e-10, 8), (B.LQ_HALF, 1e-2, 1e-9, 12),
                                                   (B.LQ_FP32, 1e-3, 1e-9, 1)])
def test_batched_bicgstab_variant(inner, delta, tol, nrhs):
    """Solver variant of SURVEY 8(f) #3: batched BiCGStab on Mhat with complex per-RHS scalars inside the same fp64 defect correction;
    same acceptance as the CG path (true residual by the oracle's M, solution against the oracle's CG) and fewer operator calls."""
    dims = (8, 8, 8, 16)
    ctx, orc = setup(dims, 1001, 0.2, 0.124, 1.2)
    b = inputs.laph_sources(dims, nrhs, 2, 2001) if nrhs >= 8 else inputs.gaussian_spinors(dims, nrhs, 2005)
    x, info = ctx.solve(b, tol=tol, inner_prec=inner, delta=delta, check_every=2, algorithm=B.LQ_ALG_BICGSTAB)
    x_cg, info_cg = ctx.solve(b, tol=tol, inner_prec=inner, delta=delta, check_every=2)
    ctx.close()
    assert info["converged"], info
    res = true_residuals(orc, x, b)
    assert np.all(res <= tol), res
    assert np.allclose(res, info["true_rel_residual"], rtol=1e-3, atol=tol * 1e-3)
    k = nrhs // 2
    xo, _, _ = oracle.solve_eo(dims, orc.U, orc.A, orc.Ainv, 0.124, b[k], tol * 1e-2)
    assert rel_err(x[k], xo.reshape(x[k].shape)) <= 50 * tol
    assert info["dslash_applies"] < info_cg["dslash_applies"]


@pytest.mark.parametrize("algorithm", [B.LQ_ALG_CGNR, B.LQ_ALG_BICGSTAB])
def test_half_solver_with_int16_links(algorithm):
    """the int16+norm inner solver with int16 links still converges to the fp64 solution (the defect correction
    uses the full-precision operator); true residual by the oracle's M."""
    dims = (8, 8, 8, 16)
    ctx, orc = setup(dims, 1003, 0.3, 0.1235, 1.0)
    ctx.set_half_links(True)
    b = inputs.laph_sources(dims, 12, 3, 2003)
    x, info = ctx.solve(b, tol=1e-9, inner_prec=B.LQ_HALF, delta=1e-2, check_every=2, use_graph=True, algorithm=algorithm)
    assert info["converged"], info
    assert np.all(true_residuals(orc, x, b) <= 1e-9)
    ctx.close()
