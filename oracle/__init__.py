"""oracle -- TEST INFRASTRUCTURE, NOT PRODUCT.

ctypes front end of `wilson_clover_oracle.c` (plain fp64 C; see that file's header for the
citations and the list of pins).  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / `--impl reference` legs may import this package; the product path
(paper_2510_26313_b200) never does.

All arrays are numpy complex128 in the canonical layouts:
    gauge  U[mu][t][z][y][x][3][3]     spinor psi[t][z][y][x][4][3]     clover A[t][z][y][x][12][12]
`dims` is always (Lx, Ly, Lz, Lt).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "wilson_clover_oracle.c")
# ORACLE_SANITIZE=1: build and load an AddressSanitizer + UndefinedBehaviorSanitizer build instead; run as
#   ORACLE_SANITIZE=1 LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0 python -m pytest tests -m "not gpu" -q
_SANITIZE = os.environ.get("ORACLE_SANITIZE", "0") == "1"
_SO = os.path.join(_HERE, "liboracle_san.so" if _SANITIZE else "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, OpenMP, no fast-math: IEEE semantics, reading #19)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        opt = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"] if _SANITIZE else ["-O2"]
        cmd = ["gcc"] + opt + ["-std=c11", "-fopenmp", "-fPIC", "-shared", "-fno-fast-math", "-o", _SO, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _SO


def _c(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_SO)
        _lib.orc_norm2.restype = ctypes.c_double
        _lib.orc_norm2.argtypes = [ctypes.c_long, ctypes.c_void_p]
        _lib.orc_clover_inverse.argtypes = [ctypes.c_long, ctypes.c_void_p, ctypes.c_void_p]
        _lib.orc_apply_site_matrix.argtypes = [ctypes.c_long, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
    return _lib


def _dims(dims):
    return (ctypes.c_int * 4)(*[int(d) for d in dims])


def _vol(dims):
    return int(dims[0]) * int(dims[1]) * int(dims[2]) * int(dims[3])


def _cc(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.complex128)
    if shape is not None:
        assert a.size == int(np.prod(shape)), (a.shape, shape)
    return a


def num_threads() -> int:
    return int(lib().orc_num_threads())


def gamma(mu: int) -> np.ndarray:
    """gamma_mu for mu in 0..3, gamma5 for mu == 5 (4x4 complex)."""
    out = np.zeros((4, 4), dtype=np.complex128)
    lib().orc_gamma(ctypes.c_int(mu), _c(out))
    return out


def sigma(mu: int, nu: int) -> np.ndarray:
    out = np.zeros((4, 4), dtype=np.complex128)
    lib().orc_sigma(ctypes.c_int(mu), ctypes.c_int(nu), _c(out))
    return out


def hop(dims, U, psi, t_bc: int = -1) -> np.ndarray:
    """D psi on the full lattice."""
    V = _vol(dims)
    U = _cc(U, (4, V, 3, 3)); psi = _cc(psi, (V, 12))
    out = np.empty_like(psi)
    lib().orc_hop(_dims(dims), ctypes.c_int(t_bc), _c(U), _c(psi), _c(out))
    return out


def field_strength(dims, U) -> np.ndarray:
    """F[plane][t][z][y][x][3][3], planes (xy, xz, xt, yz, yt, zt) (step 5)."""
    V = _vol(dims)
    U = _cc(U, (4, V, 3, 3))
    Lx, Ly, Lz, Lt = dims
    F = np.empty((6, Lt, Lz, Ly, Lx, 3, 3), dtype=np.complex128)
    lib().orc_field_strength(_dims(dims), _c(U), _c(F))
    return F


def clover(dims, U, kappa: float, csw: float) -> np.ndarray:
    """A[t][z][y][x][12][12] (step 6)."""
    V = _vol(dims)
    U = _cc(U, (4, V, 3, 3))
    Lx, Ly, Lz, Lt = dims
    A = np.empty((Lt, Lz, Ly, Lx, 12, 12), dtype=np.complex128)
    lib().orc_clover(_dims(dims), _c(U), ctypes.c_double(kappa), ctypes.c_double(csw), _c(A))
    return A


def clover_inverse(A) -> np.ndarray:
    A = _cc(A)
    Ainv = np.empty_like(A)
    rc = lib().orc_clover_inverse(ctypes.c_long(A.size // 144), _c(A), _c(Ainv))
    if rc != 0:
        raise ArithmeticError("singular clover block")
    return Ainv


def apply_site_matrix(C, psi) -> np.ndarray:
    C = _cc(C); psi = _cc(psi)
    out = np.empty_like(psi)
    lib().orc_apply_site_matrix(ctypes.c_long(psi.size // 12), _c(C), _c(psi), _c(out))
    return out


def M(dims, U, A, kappa: float, psi, dagger: bool = False, t_bc: int = -1) -> np.ndarray:
    """M psi = A psi - kappa D psi (step 7); dagger -> gamma5 M gamma5."""
    V = _vol(dims)
    U = _cc(U, (4, V, 3, 3)); A = _cc(A, (V, 144)); psi = _cc(psi, (V, 12))
    out = np.empty_like(psi)
    lib().orc_M(_dims(dims), ctypes.c_int(t_bc), _c(U), _c(A), ctypes.c_double(kappa), ctypes.c_int(int(dagger)),
                _c(psi), _c(out))
    return out


def Mhat(dims, U, A, Ainv, kappa: float, psi, dagger: bool = False, t_bc: int = -1) -> np.ndarray:
    """Even-odd Schur operator on even sites (step 8); odd sites of the result are zero."""
    V = _vol(dims)
    U = _cc(U, (4, V, 3, 3)); A = _cc(A, (V, 144)); Ainv = _cc(Ainv, (V, 144)); psi = _cc(psi, (V, 12))
    out = np.empty_like(psi)
    lib().orc_Mhat(_dims(dims), ctypes.c_int(t_bc), _c(U), _c(A), _c(Ainv), ctypes.c_double(kappa),
                   ctypes.c_int(int(dagger)), _c(psi), _c(out))
    return out


def schur_source(dims, U, Ainv, kappa: float, b, t_bc: int = -1) -> np.ndarray:
    V = _vol(dims)
    U = _cc(U, (4, V, 3, 3)); Ainv = _cc(Ainv, (V, 144)); b = _cc(b, (V, 12))
    out = np.empty_like(b)
    lib().orc_schur_source(_dims(dims), ctypes.c_int(t_bc), _c(U), _c(Ainv), ctypes.c_double(kappa), _c(b), _c(out))
    return out


def schur_reconstruct(dims, U, Ainv, kappa: float, b, x_e, t_bc: int = -1) -> np.ndarray:
    V = _vol(dims)
    U = _cc(U, (4, V, 3, 3)); Ainv = _cc(Ainv, (V, 144)); b = _cc(b, (V, 12))
    x = np.array(x_e, dtype=np.complex128, order="C", copy=True)
    lib().orc_schur_reconstruct(_dims(dims), ctypes.c_int(t_bc), _c(U), _c(Ainv), ctypes.c_double(kappa), _c(b), _c(x))
    return x


def solve_eo(dims, U, A, Ainv, kappa: float, b, tol: float, maxit: int = 10000, t_bc: int = -1):
    """Even-odd CGNR (step 9).  Returns (x_full, iterations, true relative residual)."""
    V = _vol(dims)
    U = _cc(U, (4, V, 3, 3)); A = _cc(A, (V, 144)); Ainv = _cc(Ainv, (V, 144)); b = _cc(b, (V, 12))
    x = np.zeros_like(b)
    rel = ctypes.c_double(0.0)
    it = lib().orc_solve_eo(_dims(dims), ctypes.c_int(t_bc), _c(U), _c(A), _c(Ainv), ctypes.c_double(kappa), _c(b), _c(x),
                            ctypes.c_double(tol), ctypes.c_int(maxit), ctypes.byref(rel))
    return x, int(it), float(rel.value)


def solve_full(dims, U, A, kappa: float, b, tol: float, maxit: int = 10000, t_bc: int = -1):
    """CG on the unpreconditioned normal equations (cross-check of step 9)."""
    V = _vol(dims)
    U = _cc(U, (4, V, 3, 3)); A = _cc(A, (V, 144)); b = _cc(b, (V, 12))
    x = np.zeros_like(b)
    rel = ctypes.c_double(0.0)
    it = lib().orc_solve_full(_dims(dims), ctypes.c_int(t_bc), _c(U), _c(A), ctypes.c_double(kappa), _c(b), _c(x),
                              ctypes.c_double(tol), ctypes.c_int(maxit), ctypes.byref(rel))
    return x, int(it), float(rel.value)


def site_eval(dims, kind: int, sites, kappa: float, csw: float, coef: float = 0.0, t_bc: int = -1, rhs: int = 0,
              U=None, gauge_seed: int = 0, eps: float = 0.0, psi=None, in_seed: int = 0, xin=None, x_seed: int = 0) -> np.ndarray:
    """Site-local hop (kind 0), kernel A (1) or kernel B (2) at `sites` [n][4] = (x, y, z, t) (step 12(ii)).
    Links come from the host array U or, if U is None, from the counter-based generator (gauge_seed, eps);
    the input spinor from psi (one RHS, [V][12]) or the generator (in_seed, rhs); likewise xin / x_seed for
    kernel B.  Returns out[n][4][3]."""
    V = _vol(dims)
    sites = np.ascontiguousarray(sites, dtype=np.int32).reshape(-1, 4)
    n = sites.shape[0]
    out = np.empty((n, 4, 3), dtype=np.complex128)
    Ua = _cc(U, (4, V, 3, 3)) if U is not None else None
    pa = _cc(psi, (V, 12)) if psi is not None else None
    xa = _cc(xin, (V, 12)) if xin is not None else None
    f = lib().orc_site_eval
    f.restype = ctypes.c_int
    rc = f(_dims(dims), ctypes.c_int(t_bc), ctypes.c_int(kind), ctypes.c_double(kappa), ctypes.c_double(csw), ctypes.c_double(coef),
           _c(Ua) if Ua is not None else None, ctypes.c_uint64(gauge_seed), ctypes.c_double(eps),
           _c(pa) if pa is not None else None, ctypes.c_uint64(in_seed),
           _c(xa) if xa is not None else None, ctypes.c_uint64(x_seed), ctypes.c_long(rhs),
           ctypes.c_long(n), sites.ctypes.data_as(ctypes.c_void_p), _c(out))
    if rc != 0:
        raise ArithmeticError("singular clover block")
    return out


def laplacian(dims, U, v) -> np.ndarray:
    """3-d gauge-covariant Laplacian on every time-slice: v[vec][t][z][y][x][3] -> same shape."""
    V = _vol(dims)
    U = _cc(U, (4, V, 3, 3))
    v = np.ascontiguousarray(v, dtype=np.complex128)
    nvec = v.size // (3 * V)
    out = np.empty_like(v)
    lib().orc_laplacian(_dims(dims), _c(U), ctypes.c_long(nvec), _c(v), _c(out))
    return out


def laph_eigen(dims, U, n_ev: int):
    """Lowest n_ev eigenpairs of -Laplacian on every time-slice by the plain definition: the dense
    3*Ls^3 x 3*Ls^3 matrix of each slice is assembled by applying `laplacian` to unit vectors and handed to
    numpy.linalg.eigh.  Small lattices only.  Returns (evals[Lt][n_ev] ascending, evecs[Lt][n_ev][z][y][x][3])."""
    Lx, Ly, Lz, Lt = dims
    K = 3 * Lx * Ly * Lz
    basis = np.zeros((K, Lt, Lz, Ly, Lx, 3), dtype=np.complex128)
    flat = basis.reshape(K, Lt, K)
    for k in range(K):
        flat[k, :, k] = 1.0                       # the same unit vector on every slice: slices do not couple
    cols = laplacian(dims, U, basis).reshape(K, Lt, K)
    evals = np.empty((Lt, n_ev)); evecs = np.empty((Lt, n_ev, Lz, Ly, Lx, 3), dtype=np.complex128)
    for t in range(Lt):
        A = -cols[:, t, :].T                      # A[:, k] = -Lap e_k
        w, v = np.linalg.eigh(0.5 * (A + A.conj().T))
        evals[t] = w[:n_ev]
        evecs[t] = v[:, :n_ev].T.reshape(n_ev, Lz, Ly, Lx, 3)
    return evals, evecs


def project(v, psi) -> np.ndarray:
    """Eigenvector projection: P[t][alpha][j][k] = sum_{x,c} conj(v_j(x,t,c)) psi_k(x,t,alpha,c),
    v[j][t][z][y][x][3], psi[k][t][z][y][x][4][3]; the plain definition as one einsum."""
    v = np.asarray(v, dtype=np.complex128); psi = np.asarray(psi, dtype=np.complex128)
    return np.einsum("jtzyxc,ktzyxac->tajk", v.conj(), psi)
