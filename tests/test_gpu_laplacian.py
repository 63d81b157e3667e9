"""GPU parity of the batched 3-d gauge-covariant Laplacian against the oracle: every batch width,
fp64 (<= 1e-13) and fp32 (<= 1e-5; also with 12-real links), a padded lattice, wraps in every spatial direction."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle  # noqa: E402
from paper_2510_26313_b200 import binding as B, inputs  # noqa: E402


def fields(dims, nvec, seed):
    Lx, Ly, Lz, Lt = dims
    idx = np.arange(nvec * Lt * Lz * Ly * Lx * 3, dtype=np.int64)
    return inputs.cgauss(seed, inputs.STREAM_COLORVEC, idx).reshape(nvec, Lt, Lz, Ly, Lx, 3)


def rel(a, b):
    return np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel())


@pytest.mark.parametrize("dims", [(8, 4, 4, 6), (6, 6, 2, 6), (2, 2, 2, 2), (16, 4, 8, 4)])
@pytest.mark.parametrize("nvec", [1, 2, 4, 8, 12, 16, 32])
def test_laplacian_matches_oracle(dims, nvec):
    U = inputs.make_links(dims, 61, 0.3)
    v = fields(dims, nvec, 62)
    want = oracle.laplacian(dims, U, v)
    ctx = B.Context(dims)
    ctx.load_gauge(U)
    for prec, tol in ((B.LQ_FP64, 1e-13), (B.LQ_FP32, 1e-5)):
        got = ctx.laplacian(v, prec)
        for k in range(nvec):
            assert rel(got[k], want[k]) <= tol, (dims, nvec, prec, k)
    ctx.close()


def test_laplacian_recon12_and_errors():
    dims = (8, 4, 4, 4)
    U = inputs.make_links(dims, 63, 0.3)
    v = fields(dims, 4, 64)
    want = oracle.laplacian(dims, U, v)
    ctx = B.Context(dims)
    with pytest.raises(B.LqError):
        ctx.laplacian(v, B.LQ_FP32)                    # gauge field not loaded
    ctx.load_gauge(U, recon=12)
    assert rel(ctx.laplacian(v, B.LQ_FP32), want) <= 1e-5
    with pytest.raises(B.LqError):
        ctx.laplacian(v, B.LQ_HALF)
    with pytest.raises(B.LqError):
        ctx.laplacian(v[:3], B.LQ_FP64)                # unsupported batch width
    ctx.close()
