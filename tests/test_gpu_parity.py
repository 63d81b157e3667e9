"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, same seeded inputs.

Tolerances are BASELINE.json north_star's: fp64 relative L2 <= 1e-13, fp32 operator <= 1e-5, half-storage
operator <= 3e-3, solver true residual <= requested tolerance (SURVEY.md 8(c.2) readings #10, #22).
"""
import numpy as np
import pytest

from paper_2510_26313_b200 import inputs
from paper_2510_26313_b200 import binding as B
from tests.oracle_ops import OracleCase, rel_err

pytestmark = pytest.mark.gpu

TOL = {B.LQ_FP64: 1e-13, B.LQ_FP32: 1e-5, B.LQ_HALF: 3e-3}
ALL_OPS = [B.LQ_OP_HOP, B.LQ_OP_M, B.LQ_OP_MDAG, B.LQ_OP_CLOVER, B.LQ_OP_CLOVER_INV, B.LQ_OP_HOP_EO, B.LQ_OP_HOP_OE,
           B.LQ_OP_MHAT, B.LQ_OP_MHAT_DAG, B.LQ_OP_KERNEL_A, B.LQ_OP_KERNEL_B]


def make_case(dims, seed, eps, kappa, csw, recon=18, t_bc=-1):
    U = inputs.make_links(dims, seed, eps)
    ctx = B.Context(dims)
    ctx.load_gauge(U, recon=recon, t_bc=t_bc)
    ctx.build_clover(kappa, csw)
    return ctx, OracleCase(dims, U, kappa, csw, t_bc)


def check_ops(ctx, orc, nrhs, prec, ops=ALL_OPS, seed=2000):
    psi = inputs.gaussian_spinors(orc.dims, nrhs, seed)
    psi2 = inputs.gaussian_spinors(orc.dims, nrhs, seed + 17)
    worst = 0.0
    for op in ops:
        in2 = psi2 if op == B.LQ_OP_KERNEL_B else None
        got = ctx.apply(op, psi, prec, in2=in2).astype(np.complex128)
        exp = orc.apply(op, psi, in2)
        for r in range(nrhs):
            e = rel_err(got[r], exp[r])
            assert e <= TOL[prec], (op, prec, nrhs, r, e)
            worst = max(worst, e)
        # parity ops leave the other parity exactly zero
        if op in (B.LQ_OP_HOP_EO, B.LQ_OP_MHAT, B.LQ_OP_MHAT_DAG, B.LQ_OP_KERNEL_B):
            assert np.all(got * orc.odd == 0)
        if op in (B.LQ_OP_HOP_OE, B.LQ_OP_KERNEL_A):
            assert np.all(got * orc.even == 0)
    return worst


def test_config0_all_operators_fp64():
    """configs[0]: 4^3 x 8, 1 RHS, fp64, eps 0.3, kappa 0.12, csw 1.0 (reading #16: hop, M, Mdag, Mhat, Mhat^dag...)."""
    cfg = inputs.CONFIGS[0]
    ctx, orc = make_case(cfg["dims"], cfg["gauge_seed"], cfg["eps"], cfg["kappa"], cfg["csw"])
    worst = check_ops(ctx, orc, 1, B.LQ_FP64, seed=cfg["source_seed"])
    assert worst <= 1e-13
    ctx.close()


@pytest.mark.parametrize("nrhs", [1, 2, 4, 8, 12, 16, 24, 32])
@pytest.mark.parametrize("prec", [B.LQ_FP64, B.LQ_FP32, B.LQ_HALF])
def test_multi_rhs_ragged_lattice(nrhs, prec):
    """Unequal extents (Lxh = 3: x-lines do not fill a warp; several tiles and a ragged tail), every supported N."""
    dims = (6, 4, 8, 10)
    ctx, orc = make_case(dims, 1234, 0.3, 0.124, 1.2)
    ops = ALL_OPS if nrhs in (1, 8, 12) else [B.LQ_OP_M, B.LQ_OP_MHAT_DAG, B.LQ_OP_KERNEL_A, B.LQ_OP_KERNEL_B]
    check_ops(ctx, orc, nrhs, prec, ops=ops)
    ctx.close()


@pytest.mark.parametrize("variant", [0, 1])
@pytest.mark.parametrize("nrhs,rpt", [(8, 1), (8, 2), (8, 4), (2, 1), (2, 2)])
def test_rhs_per_thread_variants(nrhs, rpt, variant):
    """Every (RHS group width, RHS per thread, register-budget variant) instantiation of the stencil kernels."""
    dims = (8, 4, 4, 6)
    ctx, orc = make_case(dims, 99, 0.3, 0.12, 1.0)
    ctx.set_tuning(dslash_variant=variant, dslash_rpt=rpt)
    for prec in (B.LQ_FP64, B.LQ_FP32, B.LQ_HALF):
        check_ops(ctx, orc, nrhs, prec, ops=[B.LQ_OP_MDAG, B.LQ_OP_KERNEL_A, B.LQ_OP_KERNEL_B])
    ctx.close()


@pytest.mark.parametrize("dims", [(8, 8, 4, 6), (16, 4, 8, 4), (32, 2, 6, 2)])
@pytest.mark.parametrize("zc", [1, 2, 0xFF])
def test_sweep_order_z_chunks(dims, zc):
    """The z-chunked sweep order (launch-order block -> site block permutation, used on large lattices so that three
    time-slices of a chunk stay in L2) together with the distance prefetch: forced chunk sizes on small lattices."""
    ctx, orc = make_case(dims, 888, 0.3, 0.124, 1.0)
    for pfd in (0, 3):
        ctx.set_tuning(dslash_variant=zc << 8, dslash_pfd=pfd)
        for nrhs, prec in ((8, B.LQ_FP32), (12, B.LQ_HALF), (4, B.LQ_FP64), (1, B.LQ_FP32)):
            check_ops(ctx, orc, nrhs, prec, ops=[B.LQ_OP_MHAT_DAG, B.LQ_OP_KERNEL_A, B.LQ_OP_KERNEL_B])
    ctx.close()


@pytest.mark.parametrize("nrhs", [1, 4, 12])
@pytest.mark.parametrize("prec", [B.LQ_FP64, B.LQ_FP32, B.LQ_HALF])
def test_l2_prefetch_distances(nrhs, prec):
    """The L2 distance prefetch must never change a result: distances smaller than, equal to and beyond the number
    of site blocks (18 here), and off."""
    dims = (6, 4, 6, 8)
    ctx, orc = make_case(dims, 555, 0.3, 0.124, 1.0)
    for pfd in (0, 1, 7, 17, 18, 500):
        ctx.set_tuning(dslash_pfd=pfd)
        check_ops(ctx, orc, nrhs, prec, ops=[B.LQ_OP_MHAT, B.LQ_OP_KERNEL_A, B.LQ_OP_KERNEL_B])
    ctx.close()


@pytest.mark.parametrize("nrhs", [1, 4, 12])
@pytest.mark.parametrize("prec", [B.LQ_FP64, B.LQ_FP32, B.LQ_HALF])
def test_padded_last_site_block(nrhs, prec):
    """Vh = 216 is not a multiple of the 32-site native block: the last block is 3/4 padding that no kernel may
    read into a result or a reduction."""
    dims = (6, 6, 2, 6)
    ctx, orc = make_case(dims, 4321, 0.3, 0.124, 1.0)
    check_ops(ctx, orc, nrhs, prec, ops=[B.LQ_OP_HOP, B.LQ_OP_M, B.LQ_OP_MHAT, B.LQ_OP_KERNEL_A, B.LQ_OP_KERNEL_B, B.LQ_OP_CLOVER_INV])
    ctx.close()


@pytest.mark.parametrize("prec", [B.LQ_FP32, B.LQ_HALF])
def test_recon12_matches_oracle_and_recon18(prec):
    """configs[4] kernel: 12-real links, third row rebuilt in-kernel, antiperiodic sign applied to the hop."""
    dims = (8, 8, 4, 8)
    U = inputs.make_links(dims, 1004, 0.3)
    orc = OracleCase(dims, U, 0.124, 1.0)
    psi = inputs.gaussian_spinors(dims, 4, 2004)
    res = {}
    for recon in (18, 12):
        ctx = B.Context(dims)
        ctx.load_gauge(U, recon=recon)
        ctx.build_clover(0.124, 1.0)
        res[recon] = ctx.apply(B.LQ_OP_KERNEL_A, psi, prec).astype(np.complex128)
        got_m = ctx.apply(B.LQ_OP_M, psi, prec).astype(np.complex128)
        assert rel_err(got_m, orc.apply(B.LQ_OP_M, psi)) <= TOL[prec]
        ctx.close()
    exp = orc.apply(B.LQ_OP_KERNEL_A, psi)
    assert rel_err(res[12], exp) <= TOL[prec] and rel_err(res[18], exp) <= TOL[prec]
    if prec == B.LQ_FP32:
        assert rel_err(res[12], res[18]) <= 1e-6


def test_periodic_time_boundary():
    dims = (4, 4, 4, 8)
    ctx, orc = make_case(dims, 1000, 0.3, 0.12, 1.0, t_bc=+1)
    check_ops(ctx, orc, 2, B.LQ_FP64, ops=[B.LQ_OP_HOP, B.LQ_OP_M, B.LQ_OP_MHAT])
    ctx.close()


def test_minimal_lattice_2to4():
    """Degenerate case: x+mu and x-mu coincide (reading #21); Lxh = 1."""
    dims = (2, 2, 2, 2)
    ctx, orc = make_case(dims, 1000, 0.3, 0.12, 1.0)
    check_ops(ctx, orc, 1, B.LQ_FP64)
    check_ops(ctx, orc, 4, B.LQ_FP32, ops=[B.LQ_OP_M, B.LQ_OP_MHAT])
    ctx.close()


def test_clover_blocks_match_oracle():
    """Row a1: the GPU-built A and A^{-1} applied to unit vectors reproduce the oracle's dense 12x12 blocks."""
    dims = (4, 4, 4, 4)
    ctx, orc = make_case(dims, 5, 0.3, 0.124, 1.2)
    V = int(np.prod(dims))
    Lx, Ly, Lz, Lt = dims
    A = orc.A.reshape(V, 12, 12)
    Ainv = orc.Ainv.reshape(V, 12, 12)
    cols = np.zeros((12, Lt, Lz, Ly, Lx, 4, 3), dtype=np.complex128)
    for j in range(12):
        cols[j, ..., j // 3, j % 3] = 1.0
    got = ctx.apply(B.LQ_OP_CLOVER, cols, B.LQ_FP64).reshape(12, V, 12)
    goti = ctx.apply(B.LQ_OP_CLOVER_INV, cols, B.LQ_FP64).reshape(12, V, 12)
    assert np.abs(got.transpose(1, 2, 0) - A).max() < 1e-14
    assert np.abs(goti.transpose(1, 2, 0) - Ainv).max() < 1e-13
    ctx.close()


def test_pack_unpack_and_device_generators():
    """Reorders are bit-exact; the device-side counter-based generators reproduce inputs.py."""
    dims = (6, 4, 4, 8)
    ctx = B.Context(dims)
    psi = inputs.gaussian_spinors(dims, 4, 31)
    nat = ctx.pack(psi, 4, B.LQ_FP64)
    assert np.array_equal(ctx.unpack(nat, 4, B.LQ_FP64), psi)
    nat32 = ctx.pack(psi, 4, B.LQ_FP32)
    assert np.array_equal(ctx.unpack(nat32, 4, B.LQ_FP32), psi.astype(np.complex64).astype(np.complex128))
    nath = ctx.pack(psi, 4, B.LQ_HALF)
    back = ctx.unpack(nath, 4, B.LQ_HALF)
    site_max = np.abs(np.stack([psi.real, psi.imag])).max(axis=(0, 6, 7))
    assert np.all(np.abs(back - psi).max(axis=(5, 6)) <= 1.01 * site_max / 32767)      # |err| <= norm/(2*32767) per real
    gen = ctx.native_empty(4, B.LQ_FP64)
    ctx.fill_spinor_random(gen, 4, B.LQ_FP64, 31)
    assert np.abs(ctx.unpack(gen, 4, B.LQ_FP64) - psi).max() < 1e-14
    # device gauge generator vs host recipe, compared through the operator (the gauge field has no read-back call)
    U = inputs.make_links(dims, 77, 0.3)
    ctx.fill_gauge_random(77, 0.3)
    h1 = ctx.apply(B.LQ_OP_HOP, psi, B.LQ_FP64)
    ctx.load_gauge(U)
    h2 = ctx.apply(B.LQ_OP_HOP, psi, B.LQ_FP64)
    assert rel_err(h1, h2) < 1e-14
    ctx.close()


def test_error_paths():
    with pytest.raises(B.LqError):
        B.Context((4, 4, 3, 8))
    ctx = B.Context((4, 4, 4, 8))
    psi = inputs.gaussian_spinors((4, 4, 4, 8), 1, 1)
    with pytest.raises(B.LqError) as e:
        ctx.apply(B.LQ_OP_HOP, psi, B.LQ_FP64)
    assert e.value.code == B.LQ_ESTATE
    ctx.load_gauge(inputs.make_links((4, 4, 4, 8), 1, 0.3))
    with pytest.raises(B.LqError) as e:
        ctx.apply(B.LQ_OP_M, psi, B.LQ_FP64)
    assert e.value.code == B.LQ_ESTATE
    with pytest.raises(B.LqError) as e:
        ctx.apply(B.LQ_OP_HOP, np.concatenate([psi] * 3), B.LQ_FP64)
    assert e.value.code == B.LQ_EINVAL
    with pytest.raises(B.LqError) as e:
        ctx.build_clover(0.12, 400.0)          # kappa*csw*F far beyond 1: a block loses positive definiteness
    assert e.value.code == B.LQ_ESINGULAR
    ctx.build_clover(0.12, 1.0)
    assert ctx.apply(B.LQ_OP_M, psi, B.LQ_FP64).shape == psi.shape
    assert ctx.launches > 0
    ctx.close()


@pytest.mark.parametrize("nrhs", [1, 2, 4, 8, 12, 16])
def test_int16_links_in_the_half_kernels(nrhs):
    """Solver variant of SURVEY 8(f) #3 (reading #13): LQ_HALF stencil kernels with int16 fixed-point links.  Against the oracle on
    the UNQUANTISED links and spinors the half-storage tolerance holds; against the oracle on links quantised the same way
    (q = rint(32767 u) / 32767) the difference is the spinor quantisation alone."""
    dims = (8, 6, 4, 6)          # Vh = 576: 18 site blocks
    ctx, orc = make_case(dims, 51, 0.3, 0.1235, 1.0)
    ctx.set_half_links(True)
    ops = [B.LQ_OP_HOP, B.LQ_OP_M, B.LQ_OP_MDAG, B.LQ_OP_MHAT, B.LQ_OP_MHAT_DAG, B.LQ_OP_KERNEL_A, B.LQ_OP_KERNEL_B]
    worst = check_ops(ctx, orc, nrhs, B.LQ_HALF, ops=ops)
    assert worst <= 3e-3
    Uq = (np.rint(orc.U.view(np.float64) * 32767.0) / 32767.0).view(np.complex128)
    orc_q = OracleCase(dims, Uq, 0.1235, 1.0)
    orc_q.A, orc_q.Ainv = orc.A, orc.Ainv                      # the clover term is built from the full-precision links
    psi = inputs.gaussian_spinors(dims, nrhs, 7)
    got = ctx.apply(B.LQ_OP_HOP, psi, B.LQ_HALF).astype(np.complex128)
    e_q = max(rel_err(got[r], orc_q.apply(B.LQ_OP_HOP, psi)[r]) for r in range(nrhs))
    e_u = max(rel_err(got[r], orc.apply(B.LQ_OP_HOP, psi)[r]) for r in range(nrhs))
    assert e_q <= 1e-4 and e_u <= 2e-4, (e_q, e_u)
    # switching back restores the fp32 links
    ctx.set_half_links(False)
    got32 = ctx.apply(B.LQ_OP_HOP, psi, B.LQ_HALF).astype(np.complex128)
    assert max(rel_err(got32[r], orc.apply(B.LQ_OP_HOP, psi)[r]) for r in range(nrhs)) <= 1e-4
    ctx.close()
