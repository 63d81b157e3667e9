"""lq_project_noalloc (include/lqcd_b200.h): the fp64 eigenvector projection with its reduction scratch in a static device array, for
callers that cannot call cudaMalloc.  Checked against the existing path lq_project(..., LQ_DEVICE, LQ_FP64) on calls in a row that
share the scratch (a large call, a smaller one that leaves stale partial sums behind it, the large one again), plus: the library
allocates nothing during the call, and sizes beyond the static scratch are refused with a message naming the limit.
Collected last on purpose (file name): the suite runs with pytest -x."""
import ctypes

import pytest

pytestmark = pytest.mark.gpu

from paper_2510_26313_b200 import binding as B  # noqa: E402

DIMS = (8, 8, 8, 16)


def fields(torch, n_ev, n_sol, seed):
    Lx, Ly, Lz, Lt = DIMS
    g = torch.Generator(device="cuda").manual_seed(seed)
    v = torch.view_as_complex(torch.randn((n_ev, Lt, Lz, Ly, Lx, 3, 2), generator=g, device="cuda", dtype=torch.float64))
    x = torch.view_as_complex(torch.randn((n_sol, Lt, Lz, Ly, Lx, 4, 3, 2), generator=g, device="cuda", dtype=torch.float64))
    return v, x


def test_noalloc_projection_matches_the_allocating_path_on_calls_in_a_row():
    import torch
    ctx = B.Context(DIMS)
    Lx, Ly, Lz, Lt = DIMS
    cases = [(24, 8, 11), (5, 3, 12), (24, 8, 11), (64, 64, 13)]          # the last one fills the static scratch exactly
    for n_ev, n_sol, seed in cases:
        v, x = fields(torch, n_ev, n_sol, seed)
        want = ctx.project(v, x, B.LQ_FP64)                               # existing path: scratch from the allocator
        out = torch.full((Lt, 4, n_ev, n_sol), float("nan"), dtype=torch.complex128, device="cuda")
        torch.cuda.synchronize()
        n_alloc = torch.cuda.memory_stats()["allocation.all.allocated"]   # the context allocates through torch's caching allocator
        launches = ctx.launches
        ctx.project_noalloc(v, x, out)
        ctx.stream.synchronize()
        assert torch.cuda.memory_stats()["allocation.all.allocated"] == n_alloc
        assert ctx.launches == launches + 2
        scale = want.abs().max().item()
        # tolerance of tests/test_gpu_projection.py for the fp64 kernel (the two paths sum in the same order)
        assert (out - want).abs().max().item() <= 1e-12 * scale * (3 * Lx * Ly * Lz) ** 0.5
    # the detector works: the existing path does allocate
    v, x = fields(torch, 5, 3, 12)
    n_alloc = torch.cuda.memory_stats()["allocation.all.allocated"]
    ctx.project(v, x, B.LQ_FP64)
    assert torch.cuda.memory_stats()["allocation.all.allocated"] > n_alloc
    ctx.close()


def test_noalloc_projection_refuses_sizes_beyond_the_static_scratch():
    import torch
    ctx = B.Context(DIMS)
    dummy = torch.zeros(16, dtype=torch.complex128, device="cuda")         # never read: the call is refused before any launch
    p = ctypes.c_void_p(dummy.data_ptr())
    launches = ctx.launches
    rc = ctx.lib.lq_project_noalloc(ctx.h, p, p, 65, p, 64)                # 16 * 1 * 4 * 65 * 64 partial sums > 4 MiB / 16 B
    assert rc == B.LQ_EINVAL
    msg = ctx.lib.lq_last_error(ctx.h).decode()
    assert "LQ_NOALLOC_SCRATCH_BYTES" in msg and "262144" in msg, msg
    assert ctx.lib.lq_project_noalloc(ctx.h, p, p, 0, p, 4) == B.LQ_EINVAL
    assert ctx.lib.lq_project_noalloc(ctx.h, None, p, 4, p, 4) == B.LQ_EINVAL
    assert ctx.launches == launches
    ctx.close()
