"""Expected results of every lq_apply operator, computed by the CPU oracle (test infrastructure)."""
import numpy as np

import oracle
from paper_2510_26313_b200 import binding as B


def parity_mask(dims):
    Lx, Ly, Lz, Lt = dims
    t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    return ((x + y + z + t) & 1)[..., None, None]


class OracleCase:
    def __init__(self, dims, U, kappa, csw, t_bc=-1):
        self.dims, self.U, self.kappa, self.csw, self.t_bc = dims, U, kappa, csw, t_bc
        self.A = oracle.clover(dims, U, kappa, csw)
        self.Ainv = oracle.clover_inverse(self.A)
        par = parity_mask(dims)
        self.even, self.odd = (par == 0), (par == 1)

    def one(self, op, psi, psi2=None):
        d, U, k, tb = self.dims, self.U, self.kappa, self.t_bc
        sh = psi.shape
        if op == B.LQ_OP_HOP:
            return oracle.hop(d, U, psi, tb).reshape(sh)
        if op == B.LQ_OP_M:
            return oracle.M(d, U, self.A, k, psi, False, tb).reshape(sh)
        if op == B.LQ_OP_MDAG:
            return oracle.M(d, U, self.A, k, psi, True, tb).reshape(sh)
        if op == B.LQ_OP_CLOVER:
            return oracle.apply_site_matrix(self.A, psi).reshape(sh)
        if op == B.LQ_OP_CLOVER_INV:
            return oracle.apply_site_matrix(self.Ainv, psi).reshape(sh)
        if op == B.LQ_OP_HOP_EO:
            return oracle.hop(d, U, psi * self.odd, tb).reshape(sh) * self.even
        if op == B.LQ_OP_HOP_OE:
            return oracle.hop(d, U, psi * self.even, tb).reshape(sh) * self.odd
        if op == B.LQ_OP_MHAT:
            return oracle.Mhat(d, U, self.A, self.Ainv, k, psi, False, tb).reshape(sh)
        if op == B.LQ_OP_MHAT_DAG:
            return oracle.Mhat(d, U, self.A, self.Ainv, k, psi, True, tb).reshape(sh)
        if op == B.LQ_OP_KERNEL_A:
            h = oracle.hop(d, U, psi * self.even, tb).reshape(sh) * self.odd
            return oracle.apply_site_matrix(self.Ainv, h).reshape(sh) * self.odd
        if op == B.LQ_OP_KERNEL_B:
            h = oracle.hop(d, U, psi2 * self.odd, tb).reshape(sh) * self.even
            return (oracle.apply_site_matrix(self.A, psi * self.even).reshape(sh) - k * k * h) * self.even
        raise ValueError(op)

    def apply(self, op, psi, psi2=None):
        return np.stack([self.one(op, psi[r], None if psi2 is None else psi2[r]) for r in range(psi.shape[0])])


def rel_err(a, b):
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))
