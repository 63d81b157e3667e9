"""oracle.multigrid -- TEST INFRASTRUCTURE, NOT PRODUCT.

Plain numpy two-level adaptive multigrid for the Wilson-clover operator M ("adaptive geometric
multi-grid solver", L164 "mixed-precision multi-grid solver"; the construction is the standard one of the paper's ref. [19]:
near-null vectors -> aggregates x chirality -> block-orthonormal prolongator P -> Galerkin coarse operator A_c = P^dag M P ->
two-grid preconditioner inside a flexible Krylov solver).  Everything is written out as dense / explicit loops over aggregates,
in fp64, in the order of the definition; only `oracle.M` (the pinned fine operator) is reused.  Small lattices only.

Conventions shared with the CUDA path (include/lqcd_b200.h, lq_mg_*):
  aggregate of site (x,y,z,t) with block (bx,by,bz,bt): a = ax + Lcx*(ay + Lcy*(az + Lcz*at)), a_mu = x_mu // b_mu, Lc = L / b;
  chirality chi = 0 for spin 0,1 and 1 for spin 2,3 (DeGrand-Rossi: gamma5 = diag(1,1,-1,-1));
  coarse degree of freedom (a, chi, k), k = index of the near-null vector; coarse vectors are arrays [Vc][2][Nv];
  the prolongator column (a, chi, k) is near-null vector k restricted to aggregate a and chirality chi, Gram-Schmidt
  orthonormalised over k = 0, 1, ... in that order (classical order, one pass repeated twice for stability).
"""
from __future__ import annotations

import numpy as np


def aggregate_index(dims, block):
    """a[t][z][y][x] = coarse site index of every fine site; returns (a, coarse dims)."""
    Lx, Ly, Lz, Lt = dims
    bx, by, bz, bt = block
    assert Lx % bx == 0 and Ly % by == 0 and Lz % bz == 0 and Lt % bt == 0
    Lc = (Lx // bx, Ly // by, Lz // bz, Lt // bt)
    t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    a = (x // bx) + Lc[0] * ((y // by) + Lc[1] * ((z // bz) + Lc[2] * (t // bt)))
    return a, Lc


def prolongator(dims, block, vecs):
    """vecs[k][t][z][y][x][4][3] (near-null vectors) -> dense P[V*12][Vc*2*Nv] with orthonormal columns."""
    Lx, Ly, Lz, Lt = dims
    V = Lx * Ly * Lz * Lt
    nv = vecs.shape[0]
    a, Lc = aggregate_index(dims, block)
    Vc = int(np.prod(Lc))
    a = a.reshape(V)
    v = np.asarray(vecs, dtype=np.complex128).reshape(nv, V, 4, 3)
    P = np.zeros((V, 4, 3, Vc, 2, nv), dtype=np.complex128)
    for ag in range(Vc):
        sites = np.nonzero(a == ag)[0]
        for chi in range(2):
            sl = slice(2 * chi, 2 * chi + 2)
            cols = [v[k, sites, sl, :].copy() for k in range(nv)]          # each [ns][2][3]
            for k in range(nv):
                for _ in range(2):                                           # Gram-Schmidt against the earlier columns, twice
                    for j in range(k):
                        cols[k] = cols[k] - np.vdot(cols[j], cols[k]) * cols[j]
                nrm = np.sqrt(np.vdot(cols[k], cols[k]).real)
                assert nrm > 0
                cols[k] = cols[k] / nrm
                P[sites, sl, :, ag, chi, k] = cols[k]
    return P.reshape(V * 12, Vc * 2 * nv), Lc


def coarse_operator(apply_M, P):
    """Galerkin coarse operator A_c = P^dag M P as a dense matrix; apply_M maps a fine vector [V*12] to M v."""
    n = P.shape[1]
    MP = np.empty_like(P)
    for c in range(n):
        MP[:, c] = apply_M(P[:, c])
    return P.conj().T @ MP


def mr_smoother(apply_M, res, steps):
    """LQ_MG_SMOOTH_MR: delta ~ M^-1 res by `steps` minimal-residual steps on M from zero."""
    x = np.zeros_like(res)
    for _ in range(steps):
        r = res - apply_M(x)
        Mr = apply_M(r)
        om = np.vdot(Mr, r) / np.vdot(Mr, Mr)
        x = x + om * r
    return x


def schur_mr_smoother(dims, U, A, Ainv, kappa, res, steps, t_bc=-1):
    """LQ_MG_SMOOTH_EO: delta ~ M^-1 res through the even-odd Schur system (steps 8-10 of the solver): Schur source, `steps`
    minimal-residual steps on Mhat delta_e = rho_e from zero, reconstruction of the odd sites.  Uses the pinned oracle operators."""
    import oracle
    V = dims[0] * dims[1] * dims[2] * dims[3]
    r = np.asarray(res, dtype=np.complex128).reshape(V, 12)
    rho = oracle.schur_source(dims, U, Ainv, kappa, r, t_bc)
    d = np.zeros_like(rho)
    for _ in range(steps):
        t = oracle.Mhat(dims, U, A, Ainv, kappa, rho, False, t_bc)
        om = np.vdot(t, rho) / np.vdot(t, t)
        d = d + om * rho
        rho = rho - om * t
    return oracle.schur_reconstruct(dims, U, Ainv, kappa, r, d, t_bc).reshape(-1)


def two_grid_preconditioner(apply_M, P, Ac, r, smooth=4, smoother=None):
    """z ~ M^-1 r: pre-smoothing from zero, coarse-grid correction with an exact coarse solve, post-smoothing of the residual
    equation.  smoother(res) -> delta ~ M^-1 res; default: `smooth` minimal-residual steps on M (mr_smoother)."""
    if smoother is None:
        def smoother(res):
            return mr_smoother(apply_M, res, smooth)
    z = smoother(r)
    z = z + P @ np.linalg.solve(Ac, P.conj().T @ (r - apply_M(z)))
    return z + smoother(r - apply_M(z))


def fgcr(apply_M, b, tol, precond=None, maxit=200, restart=16):
    """Flexible GCR for M x = b (zero start); returns (x, iterations, relative residual history)."""
    x = np.zeros_like(b)
    r = b.copy()
    bn = np.linalg.norm(b)
    hist = [1.0]
    Z, W = [], []
    for it in range(1, maxit + 1):
        z = precond(r) if precond is not None else r.copy()
        w = apply_M(z)
        for zi, wi in zip(Z, W):
            beta = np.vdot(wi, w) / np.vdot(wi, wi)
            w = w - beta * wi
            z = z - beta * zi
        alpha = np.vdot(w, r) / np.vdot(w, w)
        x = x + alpha * z
        r = r - alpha * w
        Z.append(z); W.append(w)
        if len(Z) == restart:
            Z, W = [], []
        hist.append(np.linalg.norm(r) / bn)
        if hist[-1] <= tol:
            return x, it, hist
    return x, maxit, hist
