"""CPU oracle of stage 3 ("solve the system ... then the stresses") -- TEST
INFRASTRUCTURE ONLY, same rules as the rest of ``oracle/`` (never imported by the CUDA package).

Plain definitions, no iteration, no blocking:

* ``solve``           u = K^-1 f by a sparse direct factorisation (SciPy SuperLU) of the penalised CSR
                      matrix the oracle assembled.  The CUDA path uses Jacobi-PCG instead; both must
                      agree to the accuracy the residual tolerance implies.
* ``matvec``          y = K x from the CSR triplet (scipy.sparse product).
* ``stress``          sigma(x_q) = D B(x_q) u with the literal strain-displacement matrix B (6 x 3k,
                      Voigt order xx yy zz xy yz zx, engineering shear) and the isotropic D, from the
                      oracle's own shape-function derivatives.

Pins (tests/test_oracle_stage3.py): a linear displacement field gives the constant stress D eps
exactly (linear reproduction); a column under gravity with roller sides reproduces the paper's
"theoretical" bottom stress rho g H = 2.548 MPa to a few per cent (the paper's own
code is 6.75 % off); K u = f after the solve.  Nothing here is "parity unpinned".
"""
from __future__ import annotations

import numpy as np
import scipy.sparse as sp
import scipy.sparse.linalg as spla


def csr(row_ptr, col_idx, vals, n):
    return sp.csr_matrix((np.asarray(vals), np.asarray(col_idx), np.asarray(row_ptr)), shape=(n, n))


def solve(row_ptr, col_idx, vals, f):
    """Direct solve of K u = f (K from the CSR triplet); rows without entries keep u = 0."""
    n = len(row_ptr) - 1
    K = csr(row_ptr, col_idx, vals, n).tocsc()
    empty = np.diff(np.asarray(row_ptr)) == 0
    if empty.any():                      # nodes in no support: no equation, unknown stays zero
        K = K + sp.diags(empty.astype(np.float64)).tocsc()
    u = spla.spsolve(K, np.where(empty, 0.0, np.asarray(f)))
    return u


def matvec(row_ptr, col_idx, vals, x):
    n = len(row_ptr) - 1
    return csr(row_ptr, col_idx, vals, n) @ np.asarray(x)


def elastic_D(E: float, nu: float) -> np.ndarray:
    lam = E * nu / ((1.0 + nu) * (1.0 - 2.0 * nu))
    mu = E / (2.0 * (1.0 + nu))
    D = np.zeros((6, 6))
    D[:3, :3] = lam
    D[np.arange(3), np.arange(3)] += 2.0 * mu
    D[np.arange(3, 6), np.arange(3, 6)] = mu
    return D


def stress(support, dphi, u, E: float, nu: float) -> np.ndarray:
    """sigma (M, 6) at M points from their supports (M, k), derivatives dphi (M, 3, k) and u (3N,)."""
    support = np.asarray(support)
    M, k = support.shape
    U = np.asarray(u).reshape(-1, 3)
    D = elastic_D(E, nu)
    out = np.empty((M, 6))
    for q in range(M):
        B = np.zeros((6, 3 * k))
        gx, gy, gz = dphi[q, 0], dphi[q, 1], dphi[q, 2]
        B[0, 0::3] = gx
        B[1, 1::3] = gy
        B[2, 2::3] = gz
        B[3, 0::3], B[3, 1::3] = gy, gx      # gamma_xy
        B[4, 1::3], B[4, 2::3] = gz, gy      # gamma_yz
        B[5, 0::3], B[5, 2::3] = gz, gx      # gamma_zx
        out[q] = D @ (B @ U[support[q]].reshape(-1))
    return out
