"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests and bench.py.

This module holds NONE of the method's arithmetic (no Dirac operator, no clover term, no solver);
it only states the input recipe of BASELINE.json configs[0..4] (SURVEY.md 8(c.1) steps 3 and 10,
8(c.2) readings #2, #3, #4, #17, #24, 8(d) table).  It imports neither `oracle/` nor the CUDA binding.

Counter-based generator (reading #4): every random number is a pure function of
(seed, stream, index), so the host (here), the oracle's site-local evaluator (its own C copy) and
the device-side fill kernels (their own CUDA copy) can regenerate any element independently.

    mix(z)            = SplitMix64 finaliser: z += 0x9E3779B97F4A7C15; z = (z ^ z>>30)*0xBF58476D1CE4E5B9;
                        z = (z ^ z>>27)*0x94D049BB133111EB; z ^ z>>31          (all mod 2^64)
    bits(s,st,i,w)    = mix( mix( mix(s) + st ) + 2*i + w ),  w in {0,1}
    u1 = ((bits(.,0) >> 11) + 0.5) * 2^-53  in (0,1),   u2 = (bits(.,1) >> 11) * 2^-53 in [0,1)
    cgauss(s,st,i)    = sqrt(-ln u1) * exp(2*pi*i*u2)   ~ CN(0,1)  (Re, Im ~ N(0,1/2), reading #2)

Streams: 1 gauge, 2 Gaussian spinor, 3 LapH colour-vector field, 4 gauge transformation.
Index conventions: gauge element (site i_lex, mu, row, col) -> (i_lex*4 + mu)*9 + 3*row + col;
spinor element (rhs k, site, spin, colour) -> (k*V + i_lex)*12 + 3*spin + colour;
colour-vector (timeslice tag n, spatial site j = x + Lx*(y + Ly*z), colour c) -> (n*Vs + j)*3 + c.
"""
from __future__ import annotations

import numpy as np

STREAM_GAUGE, STREAM_SPINOR, STREAM_COLORVEC, STREAM_GTRANS = 1, 2, 3, 4

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _mix(z: np.ndarray) -> np.ndarray:
    z = z.astype(np.uint64, copy=True)
    with np.errstate(over="ignore"):
        z += np.uint64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
    return z ^ (z >> np.uint64(31))


def cgauss(seed: int, stream: int, index: np.ndarray) -> np.ndarray:
    """Complex standard normal CN(0,1) for each counter in `index` (any shape, integer)."""
    idx = np.asarray(index).astype(np.uint64)
    with np.errstate(over="ignore"):
        key = _mix(_mix(np.array([seed], dtype=np.uint64)) + np.uint64(stream))
        b0 = _mix(key + np.uint64(2) * idx)
        b1 = _mix(key + np.uint64(2) * idx + np.uint64(1))
    u1 = ((b0 >> np.uint64(11)).astype(np.float64) + 0.5) * 2.0 ** -53
    u2 = (b1 >> np.uint64(11)).astype(np.float64) * 2.0 ** -53
    r = np.sqrt(-np.log(u1))
    return r * np.exp(2j * np.pi * u2)


def volume(dims) -> int:
    return int(dims[0]) * int(dims[1]) * int(dims[2]) * int(dims[3])


def project_su3_rows(W: np.ndarray) -> np.ndarray:
    """Gram-Schmidt on ROWS, third row = conj(a x b) (reading #3).  W[..., 3, 3] -> U[..., 3, 3]."""
    a = W[..., 0, :]
    b = W[..., 1, :]
    a = a / np.linalg.norm(a, axis=-1, keepdims=True)
    b = b - np.sum(np.conj(a) * b, axis=-1, keepdims=True) * a
    b = b / np.linalg.norm(b, axis=-1, keepdims=True)
    c = np.conj(np.cross(a, b))
    return np.stack([a, b, c], axis=-2)


def make_links(dims, seed: int, eps: float) -> np.ndarray:
    """U[mu][t][z][y][x][3][3] = SU(3) projection of 1 + eps*G, G_ij ~ CN(0,1) (configs[0..4])."""
    Lx, Ly, Lz, Lt = dims
    V = volume(dims)
    site = np.arange(V, dtype=np.uint64)
    out = np.empty((4, V, 3, 3), dtype=np.complex128)
    e = np.arange(9, dtype=np.uint64)
    for mu in range(4):
        idx = (site[:, None] * np.uint64(4) + np.uint64(mu)) * np.uint64(9) + e[None, :]
        G = cgauss(seed, STREAM_GAUGE, idx).reshape(V, 3, 3)
        out[mu] = project_su3_rows(np.eye(3)[None] + eps * G)
    return out.reshape(4, Lt, Lz, Ly, Lx, 3, 3)


def unit_links(dims) -> np.ndarray:
    Lx, Ly, Lz, Lt = dims
    U = np.zeros((4, Lt, Lz, Ly, Lx, 3, 3), dtype=np.complex128)
    U[..., 0, 0] = U[..., 1, 1] = U[..., 2, 2] = 1.0
    return U


def gaussian_spinors(dims, nrhs: int, seed: int) -> np.ndarray:
    """psi[rhs][t][z][y][x][spin][colour], every component ~ CN(0,1)."""
    Lx, Ly, Lz, Lt = dims
    V = volume(dims)
    idx = np.arange(nrhs * V * 12, dtype=np.uint64)
    return cgauss(seed, STREAM_SPINOR, idx).reshape(nrhs, Lt, Lz, Ly, Lx, 4, 3)


def laph_sources(dims, nrhs: int, n_t: int, seed: int, out: np.ndarray | None = None) -> np.ndarray:
    """LapH-style time/spin-diluted sources (step 10, reading #17).

    RHS k -> (t0 = (k // 4) * Lt / n_t, spin alpha = k % 4); one complex-Gaussian colour-vector field
    per source timeslice, normalised to sum |v|^2 = 1 and shared by that timeslice's four spins.
    """
    Lx, Ly, Lz, Lt = dims
    Vs = Lx * Ly * Lz
    if out is None:
        b = np.zeros((nrhs, Lt, Lz, Ly, Lx, 4, 3), dtype=np.complex128)
    else:                                         # caller-provided storage (e.g. pinned host memory), same shape
        b = out.reshape(nrhs, Lt, Lz, Ly, Lx, 4, 3)
        b[...] = 0
    for k in range(nrhs):
        n = (k // 4) % n_t
        t0 = n * Lt // n_t
        alpha = k % 4
        idx = np.uint64(n) * np.uint64(Vs * 3) + np.arange(Vs * 3, dtype=np.uint64)
        v = cgauss(seed, STREAM_COLORVEC, idx).reshape(Lz, Ly, Lx, 3)
        v = v / np.sqrt(np.sum(np.abs(v) ** 2))
        b[k, t0, :, :, :, alpha, :] = v
    return b


def random_gauge_transform(dims, seed: int) -> np.ndarray:
    """g[t][z][y][x][3][3] in SU(3), far from the identity (eps = 1)."""
    Lx, Ly, Lz, Lt = dims
    V = volume(dims)
    idx = np.arange(V * 9, dtype=np.uint64)
    G = cgauss(seed, STREAM_GTRANS, idx).reshape(V, 3, 3)
    return project_su3_rows(np.eye(3)[None] + G).reshape(Lt, Lz, Ly, Lx, 3, 3)


# BASELINE.json configs[0..4] as concrete recipes (reading #24 for kappa/csw of 2, 4)
CONFIGS = {
    0: dict(dims=(4, 4, 4, 8), nrhs=1, eps=0.3, kappa=0.12, csw=1.0, tol=1e-10, inner="fp64", recon=18,
            source="gaussian", gauge_seed=1000, source_seed=2000),
    1: dict(dims=(16, 16, 16, 32), nrhs=8, eps=0.2, kappa=0.124, csw=1.2, tol=1e-8, inner="fp32", recon=18,
            source="laph", n_t=2, gauge_seed=1001, source_seed=2001),
    2: dict(dims=(32, 32, 32, 64), nrhs=(1, 2, 4, 8, 16), eps=0.3, kappa=0.124, csw=1.0, inner="fp32", recon=18,
            source="gaussian", gauge_seed=1002, source_seed=2002),
    3: dict(dims=(48, 48, 48, 96), nrhs=12, eps=0.3, kappa=0.1235, csw=1.0, tol=1e-9, inner="half", recon=18,
            source="laph", n_t=3, gauge_seed=1003, source_seed=2003),
    4: dict(dims=(64, 64, 64, 128), nrhs=4, eps=0.3, kappa=0.124, csw=1.0, inner="fp32", recon=12,
            source="gaussian", gauge_seed=1004, source_seed=2004),
}
