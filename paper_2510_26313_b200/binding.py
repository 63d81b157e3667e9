"""Thin ctypes binding of include/lqcd_b200.h -- argument marshalling only; every step runs in the CUDA library.

PyTorch is used for device memory (the library's scratch comes from a torch-backed allocator callback) and for
the stream (torch.cuda.current_stream()).  There is no CPU fallback: if the shared library is missing, importing
the entry points raises.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
SO_PATH = os.path.join(HERE, "liblqcd_b200.so")

LQ_ALG_CGNR, LQ_ALG_BICGSTAB = 0, 1
LQ_FP64, LQ_FP32, LQ_HALF = 0, 1, 2
LQ_HOST, LQ_DEVICE = 0, 1
LQ_CANONICAL, LQ_NATIVE = 0, 1
LQ_MAX_RHS = 32
LQ_MG_SMOOTH_MR, LQ_MG_SMOOTH_EO = 0, 1
(LQ_OP_HOP, LQ_OP_M, LQ_OP_MDAG, LQ_OP_CLOVER, LQ_OP_CLOVER_INV, LQ_OP_HOP_EO, LQ_OP_HOP_OE, LQ_OP_MHAT, LQ_OP_MHAT_DAG,
 LQ_OP_KERNEL_A, LQ_OP_KERNEL_B, LQ_OP_PROBE_LOADS) = range(12)
LQ_OK, LQ_EINVAL, LQ_ESTATE, LQ_ENOMEM, LQ_ECUDA, LQ_ENOTCONVERGED, LQ_ESINGULAR = 0, -1, -2, -3, -4, -5, -6
PREC = {"fp64": LQ_FP64, "fp32": LQ_FP32, "half": LQ_HALF}

EXPORTS = ["lq_create", "lq_destroy", "lq_last_error", "lq_set_allocator", "lq_load_gauge", "lq_fill_gauge_random",
           "lq_build_clover", "lq_apply", "lq_native_bytes", "lq_pack", "lq_unpack", "lq_fill_spinor_random", "lq_solve",
           "lq_set_tuning", "lq_kernel_launches", "lq_gather_sites", "lq_native_index", "lq_fma_peak", "lq_mem_peak", "lq_set_half_links",
           "lq_laplacian", "lq_laplacian_native", "lq_cv_native_bytes", "lq_cv_fill_random", "lq_laph_eigensolve", "lq_project",
           "lq_mg_setup", "lq_mg_setup_from_vectors", "lq_mg_free", "lq_mg_restrict", "lq_mg_prolong", "lq_mg_coarse_apply", "lq_mg_vcycle",
           "lq_mg_solve", "lq_project_noalloc", "lq_project_c64"]


class SolveParam(ctypes.Structure):
    _fields_ = [("tol", ctypes.c_double), ("max_outer", ctypes.c_int), ("max_inner", ctypes.c_int), ("inner_prec", ctypes.c_int),
                ("delta", ctypes.c_double), ("check_every", ctypes.c_int), ("use_graph", ctypes.c_int),
                ("keep_direction", ctypes.c_int), ("algorithm", ctypes.c_int), ("use_x0", ctypes.c_int)]


class EigParam(ctypes.Structure):
    _fields_ = [("n_ev", ctypes.c_int), ("m", ctypes.c_int), ("cheb_degree", ctypes.c_int), ("max_restarts", ctypes.c_int),
                ("cheb_a", ctypes.c_double), ("cheb_b", ctypes.c_double), ("tol", ctypes.c_double), ("seed", ctypes.c_ulonglong)]


class EigInfo(ctypes.Structure):
    _fields_ = [("restarts", ctypes.c_int), ("converged", ctypes.c_int), ("lap_applies", ctypes.c_double),
                ("max_ritz_residual", ctypes.c_double), ("max_true_residual", ctypes.c_double), ("seconds", ctypes.c_double),
                ("seconds_ritz", ctypes.c_double), ("seconds_ortho", ctypes.c_double)]


class SolveInfo(ctypes.Structure):
    _fields_ = [("nrhs", ctypes.c_int), ("outer_cycles", ctypes.c_int), ("inner_iters", ctypes.c_int),
                ("iters", ctypes.c_int * LQ_MAX_RHS), ("true_rel_residual", ctypes.c_double * LQ_MAX_RHS),
                ("seconds", ctypes.c_double), ("dslash_applies", ctypes.c_double), ("model_bytes", ctypes.c_double),
                ("model_flops", ctypes.c_double)]


class MgParam(ctypes.Structure):
    _fields_ = [("block", ctypes.c_int * 4), ("n_vec", ctypes.c_int), ("nu_pre", ctypes.c_int), ("nu_post", ctypes.c_int), ("smoother", ctypes.c_int),
                ("coarse_iters", ctypes.c_int), ("restart", ctypes.c_int), ("setup_tol", ctypes.c_double), ("seed", ctypes.c_uint64), ("refine", ctypes.c_int)]


class MgInfo(ctypes.Structure):
    _fields_ = [("coarse_dims", ctypes.c_int * 4), ("coarse_dof", ctypes.c_longlong), ("probes", ctypes.c_int),
                ("seconds_vectors", ctypes.c_double), ("seconds_prolongator", ctypes.c_double), ("seconds_coarse_op", ctypes.c_double),
                ("bytes", ctypes.c_size_t)]


class MgSolveInfo(ctypes.Structure):
    _fields_ = [("iters", ctypes.c_int), ("outer_cycles", ctypes.c_int), ("true_rel_residual", ctypes.c_double * LQ_MAX_RHS),
                ("seconds", ctypes.c_double), ("m_applies", ctypes.c_double)]


ALLOC_FN = ctypes.CFUNCTYPE(ctypes.c_void_p, ctypes.c_size_t, ctypes.c_void_p)
FREE_FN = ctypes.CFUNCTYPE(None, ctypes.c_void_p, ctypes.c_void_p)

_lib = None


class LqError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("lqcd_b200 error %d: %s" % (code, msg))
        self.code = code


def load_library():
    """Loads liblqcd_b200.so (fails loudly if it has not been built: there is no fallback path)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(SO_PATH):
        raise ImportError("%s not found: run `python -m paper_2510_26313_b200.build` (no CPU fallback exists)" % SO_PATH)
    lib = ctypes.CDLL(SO_PATH)
    vp, ci, cd, u64 = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_uint64
    lib.lq_create.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(ci), ci, vp]
    lib.lq_destroy.argtypes = [vp]
    lib.lq_last_error.argtypes = [vp]; lib.lq_last_error.restype = ctypes.c_char_p
    lib.lq_set_allocator.argtypes = [vp, ALLOC_FN, FREE_FN, vp]
    lib.lq_load_gauge.argtypes = [vp, vp, ci, ci, ci, ci]
    lib.lq_fill_gauge_random.argtypes = [vp, u64, cd, ci, ci]
    lib.lq_build_clover.argtypes = [vp, cd, cd]
    lib.lq_set_half_links.argtypes = [vp, ci]
    lib.lq_apply.argtypes = [vp, ci, vp, vp, vp, ci, ci, ci, ci]
    lib.lq_native_bytes.argtypes = [vp, ci, ci, ci]; lib.lq_native_bytes.restype = ctypes.c_size_t
    lib.lq_pack.argtypes = [vp, vp, vp, ci, ci, ci]
    lib.lq_unpack.argtypes = [vp, vp, vp, ci, ci, ci]
    lib.lq_fill_spinor_random.argtypes = [vp, vp, ci, ci, u64, ci, ci]
    lib.lq_solve.argtypes = [vp, vp, vp, ci, ci, ci, ctypes.POINTER(SolveParam), ctypes.POINTER(SolveInfo)]
    lib.lq_set_tuning.argtypes = [vp, ci, ci, ci]
    lib.lq_gather_sites.argtypes = [vp, vp, vp, ci, ci, ctypes.c_longlong, vp]
    lib.lq_laplacian.argtypes = [vp, vp, vp, ci, ci, ci]
    lib.lq_laplacian_native.argtypes = [vp, vp, vp, ci, ci]
    lib.lq_cv_native_bytes.argtypes = [vp, ci, ci]
    lib.lq_cv_native_bytes.restype = ctypes.c_size_t
    lib.lq_cv_fill_random.argtypes = [vp, vp, ci, ci, u64]
    lib.lq_project.argtypes = [vp, vp, vp, ci, vp, ci, ci, ci]
    lib.lq_project_noalloc.argtypes = [vp, vp, vp, ci, vp, ci]
    lib.lq_project_c64.argtypes = [vp, vp, vp, ci, vp, ci, ci]
    lib.lq_laph_eigensolve.argtypes = [vp, vp, vp, ci, ctypes.POINTER(EigParam), ctypes.POINTER(EigInfo)]
    lib.lq_kernel_launches.argtypes = [vp]; lib.lq_kernel_launches.restype = ctypes.c_longlong
    szp = ctypes.POINTER(ctypes.c_size_t)
    lib.lq_native_index.argtypes = [vp, ci, ci, ci, ci, ci, ci, ci, ci, szp, szp, szp, szp]
    lib.lq_fma_peak.argtypes = [vp, ci, cd, ctypes.POINTER(cd)]
    lib.lq_mem_peak.argtypes = [vp, ci, cd, ctypes.POINTER(cd)]
    lib.lq_mg_setup.argtypes = [vp, ctypes.POINTER(MgParam), ctypes.POINTER(MgInfo)]
    lib.lq_mg_setup_from_vectors.argtypes = [vp, ctypes.POINTER(MgParam), vp, ci, ctypes.POINTER(MgInfo)]
    lib.lq_mg_free.argtypes = [vp]
    for f in (lib.lq_mg_restrict, lib.lq_mg_prolong, lib.lq_mg_coarse_apply, lib.lq_mg_vcycle):
        f.argtypes = [vp, vp, vp, ci, ci]
    lib.lq_mg_solve.argtypes = [vp, vp, vp, ci, ci, cd, ci, ctypes.POINTER(MgSolveInfo)]
    _lib = lib
    return lib


def _ptr(a):
    """Raw pointer + location of a numpy array (host) or torch tensor (host or device)."""
    if isinstance(a, np.ndarray):
        assert a.flags["C_CONTIGUOUS"]
        return ctypes.c_void_p(a.ctypes.data), LQ_HOST
    assert a.is_contiguous()
    return ctypes.c_void_p(a.data_ptr()), (LQ_DEVICE if a.is_cuda else LQ_HOST)


class Context:
    """One lattice on one GPU: the paper's 'singleton for persistent data' as an explicit handle."""

    def __init__(self, dims, device: int = 0, torch_allocator: bool = True):
        import torch
        self.torch = torch
        self.lib = load_library()
        self.dims = tuple(int(d) for d in dims)
        self.V = int(np.prod(self.dims))
        self.device = device
        torch.cuda.set_device(device)
        # a dedicated non-default stream: the legacy default stream cannot be captured into a CUDA graph
        self.stream = torch.cuda.Stream(device=device)
        self.stream.wait_stream(torch.cuda.current_stream(device))
        h = ctypes.c_void_p()
        rc = self.lib.lq_create(ctypes.byref(h), (ctypes.c_int * 4)(*self.dims), device, ctypes.c_void_p(self.stream.cuda_stream))
        if rc != 0:
            raise LqError(rc, "lq_create failed")
        self.h = h
        self._blocks = {}
        if torch_allocator:
            def _alloc(nbytes, _user):
                try:
                    t = torch.empty(int(nbytes), dtype=torch.uint8, device="cuda:%d" % device)
                except Exception:
                    return None
                self._blocks[t.data_ptr()] = t
                return t.data_ptr()

            def _free(ptr, _user):
                self._blocks.pop(ptr, None)

            self._alloc_cb, self._free_cb = ALLOC_FN(_alloc), FREE_FN(_free)
            self._check(self.lib.lq_set_allocator(self.h, self._alloc_cb, self._free_cb, None))

    # ------------------------------------------------------------------ plumbing
    def _enter(self):
        """Order the library's stream after work already queued on torch's current stream (input tensors)."""
        self.stream.wait_stream(self.torch.cuda.current_stream(self.device))

    def _check(self, rc, allow=()):
        self.torch.cuda.current_stream(self.device).wait_stream(self.stream)
        if rc != 0 and rc not in allow:
            raise LqError(rc, self.lib.lq_last_error(self.h).decode())
        return rc

    def close(self):
        if getattr(self, "h", None) is not None and self.h:
            self.lib.lq_destroy(self.h)
            self.h = None
            self._blocks.clear()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def launches(self) -> int:
        return int(self.lib.lq_kernel_launches(self.h))

    def set_tuning(self, dslash_variant=0, dslash_rpt=0, dslash_pfd=-1):
        self._check(self.lib.lq_set_tuning(self.h, dslash_variant, dslash_rpt, dslash_pfd))

    # ------------------------------------------------------------------ gauge / clover
    def load_gauge(self, U, recon: int = 18, t_bc: int = -1):
        """U: canonical [mu][t][z][y][x][3][3] complex128/complex64, numpy (host) or torch (host/device)."""
        self._enter()
        if isinstance(U, np.ndarray):
            prec = LQ_FP64 if U.dtype == np.complex128 else LQ_FP32
            U = np.ascontiguousarray(U)
        else:
            prec = LQ_FP64 if U.dtype == self.torch.complex128 else LQ_FP32
        assert (U.size if isinstance(U, np.ndarray) else U.numel()) == 4 * self.V * 9
        p, loc = _ptr(U)
        self._check(self.lib.lq_load_gauge(self.h, p, prec, loc, recon, t_bc))

    def fill_gauge_random(self, seed: int, eps: float, recon: int = 18, t_bc: int = -1):
        self._check(self.lib.lq_fill_gauge_random(self.h, seed, eps, recon, t_bc))

    def set_half_links(self, enable: bool = True):
        """int16 fixed-point links in the LQ_HALF stencil kernels (solver variant)."""
        self._check(self.lib.lq_set_half_links(self.h, int(enable)))

    def build_clover(self, kappa: float, csw: float):
        self._check(self.lib.lq_build_clover(self.h, kappa, csw))

    # ------------------------------------------------------------------ native buffers
    def native_bytes(self, nrhs: int, prec: int, parity_only: bool = False) -> int:
        return int(self.lib.lq_native_bytes(self.h, nrhs, prec, int(parity_only)))

    def native_empty(self, nrhs: int, prec: int, parity_only: bool = False):
        return self.torch.empty(self.native_bytes(nrhs, prec, parity_only), dtype=self.torch.uint8, device="cuda:%d" % self.device)

    def native_index(self, nrhs: int, prec: int, site, rhs: int, j: int):
        """(element offset in the parity block, norm offset, byte offset of the parity block, byte offset of the norm array)."""
        o = [ctypes.c_size_t() for _ in range(4)]
        x, y, z, t = (int(v) for v in site)
        rc = self.lib.lq_native_index(self.h, nrhs, prec, x, y, z, t, rhs, j, *[ctypes.byref(v) for v in o])
        if rc != 0:
            raise LqError(rc, "lq_native_index: bad argument")
        return tuple(int(v.value) for v in o)

    def fma_peak(self, mode: int = 0, ms: float = 200.0) -> float:
        """Measured FP32 FMA peak in TFLOP/s (mode 0 scalar FFMA, 1 FFMA2 with distinct operands, 2 FFMA2 with a shared operand)."""
        self._enter()
        out = ctypes.c_double()
        self._check(self.lib.lq_fma_peak(self.h, mode, ms, ctypes.byref(out)))
        return float(out.value)

    def mem_peak(self, mode: int, mbytes: float) -> float:
        """Measured read bandwidth in GB/s: mode 0 HBM (buffer much larger than L2), mode 1 L2 -> SM (buffer inside L2)."""
        self._enter()
        out = ctypes.c_double()
        self._check(self.lib.lq_mem_peak(self.h, mode, mbytes, ctypes.byref(out)))
        return float(out.value)

    def pack(self, canonical, nrhs: int, prec: int):
        self._enter()
        out = self.native_empty(nrhs, prec)
        p, loc = _ptr(canonical)
        self._check(self.lib.lq_pack(self.h, ctypes.c_void_p(out.data_ptr()), p, nrhs, prec, loc))
        return out

    def unpack(self, native, nrhs: int, prec: int) -> np.ndarray:
        self._enter()
        Lx, Ly, Lz, Lt = self.dims
        out = np.empty((nrhs, Lt, Lz, Ly, Lx, 4, 3), dtype=np.complex128)
        self._check(self.lib.lq_unpack(self.h, ctypes.c_void_p(out.ctypes.data), ctypes.c_void_p(native.data_ptr()), nrhs, prec, LQ_HOST))
        return out

    def fill_spinor_random(self, native, nrhs: int, prec: int, seed: int, parity_only: bool = False, parity: int = 0):
        self._enter()
        self._check(self.lib.lq_fill_spinor_random(self.h, ctypes.c_void_p(native.data_ptr()), nrhs, prec, seed, int(parity_only), parity))

    def gather_sites(self, native_parity_block, nrhs: int, prec: int, sites) -> np.ndarray:
        """Values of one parity block of a native device buffer at sites [n][4] = (x, y, z, t): complex128 [n][nrhs][4][3]."""
        self._enter()
        sites = np.ascontiguousarray(sites, dtype=np.int32).reshape(-1, 4)
        out = np.empty((sites.shape[0], nrhs, 24), dtype=np.float64)
        self._check(self.lib.lq_gather_sites(self.h, ctypes.c_void_p(out.ctypes.data), ctypes.c_void_p(native_parity_block.data_ptr()),
                                             nrhs, prec, sites.shape[0], ctypes.c_void_p(sites.ctypes.data)))
        return out.view(np.complex128).reshape(sites.shape[0], nrhs, 4, 3)

    # ------------------------------------------------------------------ 3-d covariant Laplacian
    def laplacian(self, v: np.ndarray, prec: int = LQ_FP64) -> np.ndarray:
        """v[vec][t][z][y][x][3] complex128 (host) -> Lap v, same shape."""
        self._enter()
        v = np.ascontiguousarray(v, dtype=np.complex128)
        out = np.empty_like(v)
        self._check(self.lib.lq_laplacian(self.h, ctypes.c_void_p(out.ctypes.data), ctypes.c_void_p(v.ctypes.data), v.shape[0], prec, LQ_HOST))
        return out

    def laph_eigensolve(self, n_ev: int, m: int, cheb_degree: int, cheb_a: float, cheb_b: float = 12.5, tol: float = 1e-10,
                        max_restarts: int = 100, seed: int = 1, want_vectors: bool = True):
        """Lowest n_ev eigenpairs of -Laplacian on every time-slice.  Returns (evals[Lt][n_ev], evecs[n_ev][t][z][y][x][3] or None, info)."""
        self._enter()
        Lx, Ly, Lz, Lt = self.dims
        prm = EigParam(n_ev, m, cheb_degree, max_restarts, cheb_a, cheb_b, tol, seed)
        info = EigInfo()
        evals = np.empty((Lt, n_ev), dtype=np.float64)
        evecs = np.empty((n_ev, Lt, Lz, Ly, Lx, 3), dtype=np.complex128) if want_vectors else None
        rc = self.lib.lq_laph_eigensolve(self.h, ctypes.c_void_p(evals.ctypes.data), ctypes.c_void_p(evecs.ctypes.data) if want_vectors else None,
                                         LQ_HOST, ctypes.byref(prm), ctypes.byref(info))
        self._check(rc, allow=(LQ_ENOTCONVERGED,))
        d = dict(converged=bool(info.converged), restarts=info.restarts, lap_applies=info.lap_applies, max_ritz_residual=info.max_ritz_residual,
                 max_true_residual=info.max_true_residual, seconds=info.seconds, seconds_ritz=info.seconds_ritz, seconds_ortho=info.seconds_ortho)
        return evals, evecs, d

    def project(self, evecs, sols, prec: int = LQ_FP64):
        """P[t][alpha][j][k] = <v_j(t), psi_k(t, alpha)>; evecs [j][t][z][y][x][3], sols [k][t][z][y][x][4][3]: complex128 numpy (host) or
        torch (device) arrays.  Returns the same kind of array, shape [Lt][4][n_ev][n_sol]."""
        self._enter()
        Lt = self.dims[3]
        n_ev, n_sol = evecs.shape[0], sols.shape[0]
        if isinstance(evecs, np.ndarray):
            evecs = np.ascontiguousarray(evecs, dtype=np.complex128); sols = np.ascontiguousarray(sols, dtype=np.complex128)
            out = np.empty((Lt, 4, n_ev, n_sol), dtype=np.complex128)
        else:
            out = self.torch.empty((Lt, 4, n_ev, n_sol), dtype=self.torch.complex128, device=evecs.device)
        pv, loc = _ptr(evecs); px, _ = _ptr(sols); po, _ = _ptr(out)
        self._check(self.lib.lq_project(self.h, po, pv, n_ev, px, n_sol, loc, prec))
        return out

    def project_c64(self, evecs, sols):
        """lq_project_c64: the tensor-core projection of complex64 fields (numpy host arrays or torch device arrays, shapes as for
        project); returns complex128 [Lt][4][n_ev][n_sol] of the same kind."""
        self._enter()
        Lt = self.dims[3]
        n_ev, n_sol = evecs.shape[0], sols.shape[0]
        if isinstance(evecs, np.ndarray):
            evecs = np.ascontiguousarray(evecs, dtype=np.complex64); sols = np.ascontiguousarray(sols, dtype=np.complex64)
            out = np.empty((Lt, 4, n_ev, n_sol), dtype=np.complex128)
        else:
            assert evecs.dtype == sols.dtype == self.torch.complex64
            out = self.torch.empty((Lt, 4, n_ev, n_sol), dtype=self.torch.complex128, device=evecs.device)
        pv, loc = _ptr(evecs); px, _ = _ptr(sols); po, _ = _ptr(out)
        self._check(self.lib.lq_project_c64(self.h, po, pv, n_ev, px, n_sol, loc))
        return out

    def project_noalloc(self, evecs, sols, out):
        """lq_project_noalloc: fp64 projection of torch DEVICE arrays into the caller's `out` [Lt][4][n_ev][n_sol] (complex128, device)
        without any device allocation by the library (static scratch, see the header for the size limit).  Asynchronous on the
        context's stream: synchronise (self.stream.synchronize()) or order later work on self.stream before reading `out`."""
        self._enter()
        n_ev, n_sol = evecs.shape[0], sols.shape[0]
        assert evecs.is_cuda and sols.is_cuda and out.is_cuda and evecs.is_contiguous() and sols.is_contiguous() and out.is_contiguous()
        assert evecs.dtype == sols.dtype == out.dtype == self.torch.complex128 and tuple(out.shape) == (self.dims[3], 4, n_ev, n_sol)
        self._check(self.lib.lq_project_noalloc(self.h, ctypes.c_void_p(out.data_ptr()), ctypes.c_void_p(evecs.data_ptr()), n_ev,
                                                ctypes.c_void_p(sols.data_ptr()), n_sol))
        return out

    def cv_native_empty(self, nvec: int, prec: int):
        return self.torch.empty(int(self.lib.lq_cv_native_bytes(self.h, nvec, prec)), dtype=self.torch.uint8, device="cuda:%d" % self.device)

    def cv_fill_random(self, native, nvec: int, prec: int, seed: int):
        self._enter()
        self._check(self.lib.lq_cv_fill_random(self.h, ctypes.c_void_p(native.data_ptr()), nvec, prec, seed))

    def laplacian_native(self, out, inp, nvec: int, prec: int):
        self._enter()
        self._check(self.lib.lq_laplacian_native(self.h, ctypes.c_void_p(out.data_ptr()), ctypes.c_void_p(inp.data_ptr()), nvec, prec))

    # ------------------------------------------------------------------ operator
    def apply_native(self, op: int, out, inp, nrhs: int, prec: int, in2=None):
        self._enter()
        self._check(self.lib.lq_apply(self.h, op, ctypes.c_void_p(out.data_ptr()), ctypes.c_void_p(inp.data_ptr()),
                                      ctypes.c_void_p(in2.data_ptr()) if in2 is not None else None, nrhs, prec, LQ_DEVICE, LQ_NATIVE))

    def apply(self, op: int, psi: np.ndarray, prec: int = LQ_FP64, in2: np.ndarray | None = None) -> np.ndarray:
        """Canonical host arrays psi[rhs][t][z][y][x][4][3]; complex128 for fp64, complex64 otherwise."""
        dt = np.complex128 if prec == LQ_FP64 else np.complex64
        psi = np.ascontiguousarray(psi, dtype=dt)
        nrhs = psi.shape[0]
        out = np.empty_like(psi)
        p2 = None
        if in2 is not None:
            in2 = np.ascontiguousarray(in2, dtype=dt)
            p2 = ctypes.c_void_p(in2.ctypes.data)
        self._check(self.lib.lq_apply(self.h, op, ctypes.c_void_p(out.ctypes.data), ctypes.c_void_p(psi.ctypes.data), p2, nrhs, prec,
                                      LQ_HOST, LQ_CANONICAL))
        return out

    # ------------------------------------------------------------------ two-level multigrid (lq_mg_*)
    def mg_setup(self, block, n_vec: int, nu_pre: int = 2, nu_post: int = 2, coarse_iters: int = 8, restart: int = 8,
                 setup_tol: float = 1e-3, seed: int = 1, vecs=None, smoother: int = 1, refine: int = 0) -> dict:
        """Builds the hierarchy: adaptively (vecs=None) or from n_vec given canonical complex128 near-null vectors."""
        self._enter()
        prm = MgParam((ctypes.c_int * 4)(*block), n_vec, nu_pre, nu_post, smoother, coarse_iters, restart, setup_tol, seed, refine)
        info = MgInfo()
        if vecs is None:
            self._check(self.lib.lq_mg_setup(self.h, ctypes.byref(prm), ctypes.byref(info)))
        else:
            if isinstance(vecs, np.ndarray):
                vecs = np.ascontiguousarray(vecs, dtype=np.complex128)
            assert vecs.shape[0] == n_vec
            pv, loc = _ptr(vecs)
            self._check(self.lib.lq_mg_setup_from_vectors(self.h, ctypes.byref(prm), pv, loc, ctypes.byref(info)))
        self._mg = dict(coarse_dims=tuple(info.coarse_dims), n_vec=n_vec)
        return dict(coarse_dims=tuple(info.coarse_dims), coarse_dof=info.coarse_dof, probes=info.probes, seconds_vectors=info.seconds_vectors,
                    seconds_prolongator=info.seconds_prolongator, seconds_coarse_op=info.seconds_coarse_op, bytes=info.bytes)

    def mg_free(self):
        self._enter()
        self._check(self.lib.lq_mg_free(self.h))

    def _mg_piece(self, fn, inp: np.ndarray, out_fine: bool) -> np.ndarray:
        self._enter()
        inp = np.ascontiguousarray(inp, dtype=np.complex128)
        nrhs = inp.shape[0]
        Lc = self._mg["coarse_dims"]
        if out_fine:
            out = np.empty((nrhs, self.dims[3], self.dims[2], self.dims[1], self.dims[0], 4, 3), dtype=np.complex128)
        else:
            out = np.empty((nrhs, int(np.prod(Lc)), 2, self._mg["n_vec"]), dtype=np.complex128)
        self._check(fn(self.h, ctypes.c_void_p(out.ctypes.data), ctypes.c_void_p(inp.ctypes.data), nrhs, LQ_HOST))
        return out

    def mg_restrict(self, fine: np.ndarray) -> np.ndarray:
        """coarse[rhs][a][chi][k] = P^dag fine (canonical complex128 fine vectors)."""
        return self._mg_piece(self.lib.lq_mg_restrict, fine, False)

    def mg_prolong(self, coarse: np.ndarray) -> np.ndarray:
        return self._mg_piece(self.lib.lq_mg_prolong, coarse, True)

    def mg_coarse_apply(self, coarse: np.ndarray) -> np.ndarray:
        return self._mg_piece(self.lib.lq_mg_coarse_apply, coarse, False)

    def mg_vcycle(self, r: np.ndarray) -> np.ndarray:
        return self._mg_piece(self.lib.lq_mg_vcycle, r, True)

    def mg_solve(self, b, tol: float, max_iter: int = 200, x_out=None):
        """Solves M x = b with the multigrid-preconditioned flexible GCR.  b: canonical complex128 (numpy or torch, host or device)."""
        self._enter()
        if isinstance(b, np.ndarray):
            b = np.ascontiguousarray(b, dtype=np.complex128)
            x = x_out if x_out is not None else np.empty_like(b)
        else:
            x = x_out if x_out is not None else self.torch.empty_like(b)
        nrhs = b.shape[0]
        pb, loc = _ptr(b)
        px, locx = _ptr(x)
        assert loc == locx
        info = MgSolveInfo()
        rc = self.lib.lq_mg_solve(self.h, px, pb, nrhs, loc, tol, max_iter, ctypes.byref(info))
        self._check(rc, allow=(LQ_ENOTCONVERGED,))
        return x, dict(converged=(rc == 0), iters=info.iters, outer_cycles=info.outer_cycles, seconds=info.seconds, m_applies=info.m_applies,
                       true_rel_residual=list(info.true_rel_residual)[:nrhs])

    # ------------------------------------------------------------------ solve
    def solve(self, b, tol: float, inner_prec: int = LQ_FP32, delta: float = 1e-3, max_outer: int = 50, max_inner: int = 2000,
              check_every: int = 10, use_graph: bool = False, x_out=None, native: bool = False, nrhs: int | None = None,
              keep_direction: bool = True, algorithm: int = 0, use_x0: bool = False):
        """Solves M x = b.  b: canonical complex128 numpy / torch array (host or device), or a native fp64 device
        buffer when native=True (then nrhs is required).  use_x0: x_out holds the initial guess.  Returns (x, info dict)."""
        self._enter()
        prm = SolveParam(tol, max_outer, max_inner, inner_prec, delta, check_every, int(use_graph), int(keep_direction), int(algorithm), int(use_x0))
        info = SolveInfo()
        if native:
            x = x_out if x_out is not None else self.native_empty(nrhs, LQ_FP64)
            rc = self.lib.lq_solve(self.h, ctypes.c_void_p(x.data_ptr()), ctypes.c_void_p(b.data_ptr()), nrhs, LQ_DEVICE, LQ_NATIVE,
                                   ctypes.byref(prm), ctypes.byref(info))
        else:
            if isinstance(b, np.ndarray):
                b = np.ascontiguousarray(b, dtype=np.complex128)
                x = x_out if x_out is not None else np.empty_like(b)
            else:
                x = x_out if x_out is not None else self.torch.empty_like(b)
            nrhs = b.shape[0]
            pb, loc = _ptr(b)
            px, locx = _ptr(x)
            assert loc == locx
            rc = self.lib.lq_solve(self.h, px, pb, nrhs, loc, LQ_CANONICAL, ctypes.byref(prm), ctypes.byref(info))
        self._check(rc, allow=(LQ_ENOTCONVERGED,))
        d = dict(converged=(rc == 0), nrhs=info.nrhs, outer_cycles=info.outer_cycles, inner_iters=info.inner_iters,
                 iters=list(info.iters)[:nrhs], true_rel_residual=list(info.true_rel_residual)[:nrhs], seconds=info.seconds,
                 dslash_applies=info.dslash_applies, model_bytes=info.model_bytes, model_flops=info.model_flops)
        return x, d
