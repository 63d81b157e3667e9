"""Out-of-bounds checks of our own (compute-sanitizer is closed on this GPU pool): every native buffer handed to the library
sits between guard bands.  Guard bands of INPUTS hold NaN (int16: norm NaN), so a read outside a buffer poisons the result;
guard bands of OUTPUTS hold a sentinel byte pattern that must survive.  Results must also equal, bit for bit, those obtained
with plain (unguarded) buffers.  Lattices include a padded last site block and a minimal 2^4 lattice."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from paper_2510_26313_b200 import binding as B, inputs  # noqa: E402

GUARD = 1 << 16        # bytes on each side (multiple of 256)


class Guarded:
    """A device buffer of `nbytes` between two guard bands filled with `fill` (a uint8 pattern or NaN floats)."""

    def __init__(self, nbytes, nan_guard):
        self.n = nbytes
        self.raw = torch.empty(nbytes + 2 * GUARD, dtype=torch.uint8, device="cuda")
        if nan_guard:
            self.raw.view(torch.float32)[:] = float("nan")     # 0x7FC00000: as int16 pairs (0x0000, 0x7FC0) -- the norm guard decides
        else:
            self.raw[:] = 0xA5
        self.buf = self.raw[GUARD:GUARD + nbytes]
        assert self.buf.data_ptr() % 256 == 0

    def guards_intact(self, value=0xA5):
        return bool((self.raw[:GUARD] == value).all()) and bool((self.raw[GUARD + self.n:] == value).all())


@pytest.mark.parametrize("dims", [(6, 6, 2, 2), (2, 2, 2, 2), (8, 4, 4, 6), (12, 6, 2, 4)])
@pytest.mark.parametrize("prec", [B.LQ_FP64, B.LQ_FP32, B.LQ_HALF])
@pytest.mark.parametrize("nrhs", [1, 8, 12])
def test_stencil_kernels_stay_inside_their_buffers(dims, prec, nrhs):
    ctx = B.Context(dims)
    ctx.load_gauge(inputs.make_links(dims, 11, 0.3), recon=18)
    ctx.build_clover(0.12, 1.0)
    nb = ctx.native_bytes(nrhs, prec, True)
    # plain buffers
    x = ctx.native_empty(nrhs, prec, True); y = ctx.native_empty(nrhs, prec, True)
    x.zero_(); y.zero_()
    ctx.fill_spinor_random(x, nrhs, prec, 5, parity_only=True, parity=0)
    ctx.fill_spinor_random(y, nrhs, prec, 6, parity_only=True, parity=1)
    ref = {}
    for name, op, args in (("A", B.LQ_OP_KERNEL_A, (x,)), ("B", B.LQ_OP_KERNEL_B, (x, y)), ("hop", B.LQ_OP_HOP_OE, (x,)), ("mhat", B.LQ_OP_MHAT, (x,)),
                           ("mhatdag", B.LQ_OP_MHAT_DAG, (x,))):
        out = ctx.native_empty(nrhs, prec, True)
        out.zero_()
        ctx.apply_native(op, out, args[0], nrhs, prec, in2=args[1] if len(args) > 1 else None)
        torch.cuda.synchronize()
        ref[name] = out.clone()
    # guarded buffers: inputs between NaN bands, outputs between sentinel bands
    gx, gy = Guarded(nb, True), Guarded(nb, True)
    gx.buf.copy_(x); gy.buf.copy_(y)
    for name, op, two in (("A", B.LQ_OP_KERNEL_A, False), ("B", B.LQ_OP_KERNEL_B, True), ("hop", B.LQ_OP_HOP_OE, False), ("mhat", B.LQ_OP_MHAT, False),
                          ("mhatdag", B.LQ_OP_MHAT_DAG, False)):
        go = Guarded(nb, False)
        go.buf.zero_()
        ctx.apply_native(op, go.buf, gx.buf, nrhs, prec, in2=gy.buf if two else None)
        torch.cuda.synchronize()
        assert go.guards_intact(), (name, "wrote outside the output buffer")
        assert torch.equal(go.buf, ref[name]), (name, "result differs from the unguarded run: a read went outside an input buffer")
    ctx.close()


@pytest.mark.parametrize("inner", [B.LQ_FP32, B.LQ_HALF])
@pytest.mark.parametrize("algorithm", [B.LQ_ALG_CGNR, B.LQ_ALG_BICGSTAB])
def test_native_solve_stays_inside_its_buffers(inner, algorithm):
    dims, nrhs = (6, 6, 2, 4), 12                        # Vh = 144: the last site block is padded
    ctx = B.Context(dims)
    ctx.load_gauge(inputs.make_links(dims, 12, 0.25))
    ctx.build_clover(0.124, 1.1)
    b = inputs.laph_sources(dims, nrhs, 2, 13)
    nb64 = ctx.native_bytes(nrhs, B.LQ_FP64)
    plain_b = ctx.pack(b, nrhs, B.LQ_FP64)
    kw = dict(tol=1e-9, inner_prec=inner, delta=1e-2, check_every=2, use_graph=True, algorithm=algorithm, native=True, nrhs=nrhs)
    plain_x, info = ctx.solve(plain_b, **kw)
    assert info["converged"]
    gb, gx = Guarded(nb64, True), Guarded(nb64, False)
    gb.buf.copy_(plain_b)
    x2, info2 = ctx.solve(gb.buf, x_out=gx.buf, **kw)
    torch.cuda.synchronize()
    assert info2["converged"] and gx.guards_intact()
    # padding sites of the last block are unspecified: compare through the canonical layout
    assert np.array_equal(ctx.unpack(gx.buf, nrhs, B.LQ_FP64), ctx.unpack(plain_x, nrhs, B.LQ_FP64))
    ctx.close()
