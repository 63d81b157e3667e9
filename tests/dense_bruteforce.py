"""Dense brute-force construction of the Wilson-clover matrix on tiny lattices (numpy, index loops).

Independent of oracle/ and of the CUDA path: the hop is assembled block by block into a dense
(12V x 12V) matrix and the clover leaves are products along explicitly walked paths.  Used as the
"dense-matrix brute force on a 2^4 lattice" pin of BASELINE.json north_star.
"""
import numpy as np

I4 = np.eye(4)
# SURVEY.md 8(c.1) step 2 (DeGrand-Rossi), rows as printed there
GAMMA = [
    np.array([[0, 0, 0, 1j], [0, 0, 1j, 0], [0, -1j, 0, 0], [-1j, 0, 0, 0]]),
    np.array([[0, 0, 0, -1], [0, 0, 1, 0], [0, 1, 0, 0], [-1, 0, 0, 0]], dtype=complex),
    np.array([[0, 0, 1j, 0], [0, 0, 0, -1j], [-1j, 0, 0, 0], [0, 1j, 0, 0]]),
    np.array([[0, 0, 1, 0], [0, 0, 0, 1], [1, 0, 0, 0], [0, 1, 0, 0]], dtype=complex),
]
GAMMA5 = np.diag([1.0, 1.0, -1.0, -1.0]).astype(complex)


def coords(i, dims):
    x = i % dims[0]; i //= dims[0]
    y = i % dims[1]; i //= dims[1]
    z = i % dims[2]; i //= dims[2]
    return [x, y, z, i]


def index(c, dims):
    return c[0] + dims[0] * (c[1] + dims[1] * (c[2] + dims[2] * c[3]))


def link(U, mu, c):
    """U is canonical [mu][t][z][y][x][3][3]."""
    return U[mu, c[3], c[2], c[1], c[0]]


def dense_hop(dims, U, t_bc=-1):
    V = int(np.prod(dims))
    D = np.zeros((12 * V, 12 * V), dtype=complex)
    for i in range(V):
        c = coords(i, dims)
        for mu in range(4):
            cf = list(c); cf[mu] = (c[mu] + 1) % dims[mu]
            sgn = t_bc if (mu == 3 and c[3] == dims[3] - 1) else 1
            j = index(cf, dims)
            D[12 * i:12 * i + 12, 12 * j:12 * j + 12] += sgn * np.kron(I4 - GAMMA[mu], link(U, mu, c))
            cb = list(c); cb[mu] = (c[mu] - 1) % dims[mu]
            sgn = t_bc if (mu == 3 and c[3] == 0) else 1
            j = index(cb, dims)
            D[12 * i:12 * i + 12, 12 * j:12 * j + 12] += sgn * np.kron(I4 + GAMMA[mu], link(U, mu, cb).conj().T)
    return D


def walk(dims, U, c, steps):
    """Ordered product of links along a path starting at c; step = (mu, +1|-1)."""
    c = list(c)
    P = np.eye(3, dtype=complex)
    for mu, d in steps:
        if d > 0:
            P = P @ link(U, mu, c)
            c[mu] = (c[mu] + 1) % dims[mu]
        else:
            c[mu] = (c[mu] - 1) % dims[mu]
            P = P @ link(U, mu, c).conj().T
    return P, c


def field_strength_site(dims, U, c, mu, nu):
    leaves = [
        [(mu, 1), (nu, 1), (mu, -1), (nu, -1)],
        [(nu, 1), (mu, -1), (nu, -1), (mu, 1)],
        [(mu, -1), (nu, -1), (mu, 1), (nu, 1)],
        [(nu, -1), (mu, 1), (nu, 1), (mu, -1)],
    ]
    Q = np.zeros((3, 3), dtype=complex)
    for steps in leaves:
        P, end = walk(dims, U, c, steps)
        assert end == list(c)
        Q += P
    return (Q - Q.conj().T) / 8j


def dense_clover(dims, U, kappa, csw):
    V = int(np.prod(dims))
    A = np.zeros((12 * V, 12 * V), dtype=complex)
    for i in range(V):
        c = coords(i, dims)
        blk = np.eye(12, dtype=complex)
        for mu in range(4):
            for nu in range(mu + 1, 4):
                sig = 0.5j * (GAMMA[mu] @ GAMMA[nu] - GAMMA[nu] @ GAMMA[mu])
                blk -= kappa * csw * np.kron(sig, field_strength_site(dims, U, c, mu, nu))
        A[12 * i:12 * i + 12, 12 * i:12 * i + 12] = blk
    return A


def dense_M(dims, U, kappa, csw, t_bc=-1):
    return dense_clover(dims, U, kappa, csw) - kappa * dense_hop(dims, U, t_bc)


def parity_vector(dims):
    V = int(np.prod(dims))
    return np.array([sum(coords(i, dims)) & 1 for i in range(V)])
