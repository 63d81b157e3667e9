"""Boundary checks through the C ABI: a NATIVE buffer built from the header's description alone, the
lq_native_index helper, the initial guess (use_x0), the modelled bytes / flops of lq_solve_info, and the degenerate BiCGStab
batch.  Expected operator values come from the oracle."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

import oracle  # noqa: E402
from paper_2510_26313_b200 import binding as B, inputs  # noqa: E402
from tests.oracle_ops import OracleCase, rel_err  # noqa: E402


def header_native_layout(dims, psi, prec):
    """Full-lattice native buffer written ONLY from the text of include/lqcd_b200.h ("NATIVE spinor layout"): groups of R right-hand
    sides, blocks of 32 checkerboard sites, payload[blk][g][j][s][r], norms[blk][g][s][r], parity blocks padded to 256 bytes."""
    Lx, Ly, Lz, Lt = dims
    N = psi.shape[0]
    R = 4 if N % 4 == 0 else (2 if N % 2 == 0 else 1)
    G = N // R
    Vh = Lx * Ly * Lz * Lt // 2
    NB = (Vh + 31) // 32
    dt = {B.LQ_FP64: np.float64, B.LQ_FP32: np.float32, B.LQ_HALF: np.int16}[prec]
    t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    par = (x + y + z + t) & 1
    cb = x // 2 + (Lx // 2) * (y + Ly * (z + Lz * t))
    reals = np.ascontiguousarray(psi).view(np.float64).reshape(N, Lt, Lz, Ly, Lx, 24)      # j = 2*(3*spin+colour) + re/im
    blocks = []
    for p in (0, 1):
        pay = np.zeros((NB, G, 24, 32, R), dtype=dt)
        nrm = np.zeros((NB, G, 32, R), dtype=np.float32)
        m = par == p
        c = cb[m]
        for k in range(N):
            v = reals[k][m]                                         # [Vh][24]
            if prec == B.LQ_HALF:
                n = np.max(np.abs(v.astype(np.float32)), axis=1)
                q = np.rint(v.astype(np.float32) * (np.float32(32767.0) / np.where(n > 0, n, 1))[:, None])
                nrm[c // 32, k // R, c % 32, k % R] = n
                pay[c // 32, k // R, :, c % 32, k % R] = q.astype(np.int16)
            else:
                pay[c // 32, k // R, :, c % 32, k % R] = v.astype(dt)
        raw = pay.tobytes()
        raw += b"\0" * (-len(raw) % 256)
        if prec == B.LQ_HALF:
            nb = nrm.tobytes()
            raw += nb + b"\0" * (-len(nb) % 256)
        blocks.append(raw)
    return np.frombuffer(b"".join(blocks), dtype=np.uint8).copy()


@pytest.mark.parametrize("dims,nrhs", [((8, 8, 4, 8), 8), ((6, 4, 4, 4), 2), ((4, 6, 2, 4), 1), ((8, 4, 4, 8), 12)])
@pytest.mark.parametrize("prec,tol", [(B.LQ_FP64, 1e-13), (B.LQ_FP32, 1e-5), (B.LQ_HALF, 3e-3)])
def test_native_buffer_built_from_the_header(dims, nrhs, prec, tol):
    U = inputs.make_links(dims, 21, 0.3)
    ctx = B.Context(dims)
    ctx.load_gauge(U)
    ctx.build_clover(0.12, 1.0)
    orc = OracleCase(dims, U, 0.12, 1.0)
    psi = inputs.gaussian_spinors(dims, nrhs, 22)
    host = header_native_layout(dims, psi, prec)
    assert host.size == ctx.native_bytes(nrhs, prec)
    nin = torch.from_numpy(host).cuda()
    nout = ctx.native_empty(nrhs, prec)
    ctx.apply_native(B.LQ_OP_M, nout, nin, nrhs, prec)
    got = ctx.unpack(nout, nrhs, prec)
    exp = orc.apply(B.LQ_OP_M, psi)
    assert rel_err(got, exp) <= tol
    # the packer of the library writes the same bytes as the header's description (padding sites excluded: fp64 / fp32 only)
    if prec != B.LQ_HALF and (np.prod(dims) // 2) % 32 == 0:
        assert np.array_equal(ctx.pack(psi, nrhs, prec).cpu().numpy(), host)
    # lq_native_index agrees with the formula of the header
    rng = np.random.default_rng(5)
    esz = {B.LQ_FP64: 8, B.LQ_FP32: 4, B.LQ_HALF: 2}[prec]
    view = {B.LQ_FP64: np.float64, B.LQ_FP32: np.float32, B.LQ_HALF: np.int16}[prec]
    for _ in range(50):
        site = [int(rng.integers(0, d)) for d in dims]
        k, j = int(rng.integers(0, nrhs)), int(rng.integers(0, 24))
        eo, no, pb, na = ctx.native_index(nrhs, prec, site, k, j)
        val = host[pb + eo * esz: pb + (eo + 1) * esz].view(view)[0]
        ref = psi[k, site[3], site[2], site[1], site[0]].reshape(12).view(np.float64)[j]
        if prec == B.LQ_HALF:
            nrm = host[pb + na + 4 * no: pb + na + 4 * no + 4].view(np.float32)[0]
            assert abs(float(val) * float(nrm) / 32767.0 - ref) <= 1.01 * float(nrm) / 32767.0
        else:
            assert float(val) == view(ref)
    ctx.close()


@pytest.mark.parametrize("algorithm", [B.LQ_ALG_CGNR, B.LQ_ALG_BICGSTAB])
def test_initial_guess_use_x0(algorithm):
    """use_x0: a good initial guess is honoured (fewer iterations, same solution); a wrong one does not change the answer."""
    dims = (8, 8, 8, 8)
    U = inputs.make_links(dims, 31, 0.25)
    ctx = B.Context(dims)
    ctx.load_gauge(U)
    ctx.build_clover(0.124, 1.1)
    orc = OracleCase(dims, U, 0.124, 1.1)
    b = inputs.gaussian_spinors(dims, 4, 32)
    x_ref, i_ref = ctx.solve(b, tol=1e-9, inner_prec=B.LQ_FP32, check_every=2, algorithm=algorithm)
    assert i_ref["converged"]
    # start from the converged solution: nothing left to do
    x1, i1 = ctx.solve(b, tol=1e-9, inner_prec=B.LQ_FP32, check_every=2, algorithm=algorithm, x_out=x_ref.copy(), use_x0=True)
    assert i1["converged"] and i1["inner_iters"] == 0 and i1["outer_cycles"] == 0
    assert rel_err(x1, x_ref) <= 1e-12
    # start from a perturbed solution: fewer iterations than from zero
    x0 = x_ref * (1 + 1e-4)
    x2, i2 = ctx.solve(b, tol=1e-9, inner_prec=B.LQ_FP32, check_every=2, algorithm=algorithm, x_out=x0, use_x0=True)
    assert i2["converged"] and 0 < i2["inner_iters"] < i_ref["inner_iters"]
    # start from garbage: same answer, residual by the oracle's M
    x3, i3 = ctx.solve(b, tol=1e-9, inner_prec=B.LQ_FP32, check_every=2, algorithm=algorithm, x_out=inputs.gaussian_spinors(dims, 4, 33), use_x0=True)
    assert i3["converged"]
    for x in (x2, x3):
        for k in range(4):
            r = b[k].ravel() - oracle.M(dims, U, orc.A, 0.124, x[k]).ravel()
            assert np.linalg.norm(r) / np.linalg.norm(b[k].ravel()) <= 1e-9
    # the same with device buffers
    xd, i4 = ctx.solve(torch.from_numpy(b).cuda(), tol=1e-9, inner_prec=B.LQ_FP32, check_every=2, algorithm=algorithm,
                       x_out=torch.from_numpy(x0).cuda(), use_x0=True)
    assert np.array_equal(xd.cpu().numpy(), x2)
    ctx.close()


def test_solve_info_model_counts():
    """Modelled bytes / flops (SURVEY 8(b) solve row, 8(d) byte model): the stencil part of the count follows from the number of
    stencil launches that did work; totals are positive, finite and grow with the batch."""
    dims = (8, 8, 8, 16)
    U = inputs.make_links(dims, 41, 0.2)
    ctx = B.Context(dims)
    ctx.load_gauge(U)
    ctx.build_clover(0.124, 1.2)
    Vh = np.prod(dims) // 2
    out = {}
    for n in (4, 8):
        b = inputs.laph_sources(dims, n, 2, 42)
        for use_graph in (False, True, True):
            _, info = ctx.solve(b, tol=1e-8, inner_prec=B.LQ_FP32, delta=1e-3, check_every=4, use_graph=use_graph)
            assert info["converged"]
            it, cyc = info["inner_iters"], info["outer_cycles"]
            # fp32 inner stencil launches: 4 per iteration + 2 per cycle (+2 with the direction-keeping refresh after the first)
            lo = 4 * it * Vh * n * (1320 + 504)
            assert info["model_flops"] >= lo and info["model_flops"] <= 3 * lo
            inner_bytes = it * Vh * n * (2 * (192 + 864 / n) + (288 + 864 / n) + (384 + 864 / n) + 5 * 96)
            assert info["model_bytes"] >= inner_bytes and info["model_bytes"] <= 3 * inner_bytes
            out.setdefault(n, []).append((info["model_bytes"], info["model_flops"], it))
        assert out[n][0] == out[n][1] == out[n][2]                 # the count does not depend on graph replay
    assert out[8][0][0] > out[4][0][0]
    ctx.close()


def test_bicgstab_zero_and_tiny_sources():
    """The BiCGStab path with an identically zero right-hand side (and a tiny one): the guarded divisions keep it at zero."""
    dims = (4, 4, 4, 8)
    U = inputs.make_links(dims, 1000, 0.3)
    ctx = B.Context(dims)
    ctx.load_gauge(U)
    ctx.build_clover(0.12, 1.0)
    A = oracle.clover(dims, U, 0.12, 1.0)
    b = inputs.gaussian_spinors(dims, 4, 5)
    b[1] = 0
    b[2] *= 1e-12
    for inner in (B.LQ_FP32, B.LQ_HALF):
        x, info = ctx.solve(b, tol=1e-9, inner_prec=inner, algorithm=B.LQ_ALG_BICGSTAB, check_every=2, delta=1e-2)
        assert info["converged"] and np.all(np.isfinite(x.view(np.float64)))
        assert np.all(x[1] == 0)
        res = [np.linalg.norm(b[k].ravel() - oracle.M(dims, U, A, 0.12, x[k]).ravel()) / np.linalg.norm(b[k].ravel()) for k in (0, 2, 3)]
        assert max(res) <= 1e-9
    ctx.close()


def test_clover_rebuild_failure_invalidates_the_context():
    """a failed lq_build_clover must not leave the context claiming a valid clover term."""
    dims = (4, 4, 4, 4)
    ctx = B.Context(dims)
    ctx.load_gauge(inputs.make_links(dims, 3, 0.3))
    ctx.build_clover(0.12, 1.0)
    psi = inputs.gaussian_spinors(dims, 1, 4)
    ctx.apply(B.LQ_OP_M, psi, B.LQ_FP64)
    with pytest.raises(B.LqError) as e:
        ctx.build_clover(0.12, 400.0)                               # A = 1 - kappa*csw*sigma.F is far from positive definite
    assert e.value.code == B.LQ_ESINGULAR
    with pytest.raises(B.LqError) as e:
        ctx.apply(B.LQ_OP_M, psi, B.LQ_FP64)
    assert e.value.code == B.LQ_ESTATE
    ctx.build_clover(0.12, 1.0)
    ctx.apply(B.LQ_OP_M, psi, B.LQ_FP64)
    ctx.close()
