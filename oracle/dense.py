"""Tier 0 - the definition, by dense inversion.

TEST INFRASTRUCTURE (see oracle/__init__.py).
  G^R  = (z S - H - Sigma^R_B - Sigma^R_S)^-1         PAPER.md:56, Eq. 1
  G^A  = (G^R)^H
  G^<> = G^R (Sigma^<>_B + Sigma^<>_S) G^A            PAPER.md:58, Eq. 2 solved for C^<>
restricted afterwards to blocks (i,i), (i,i+1), (i+1,i).
"""
import numpy as np

from .assemble import bt_to_dense, dagger, dense_to_bt


def gauss_jordan_inverse(M):
    """Inverse by Gauss-Jordan elimination with partial pivoting in M's own dtype.
    Exists because LAPACK has no extended precision: used with np.clongdouble (80-bit)
    for the configs[0] check (SURVEY.md 8(c) pin P1).  O(N) Python steps, vectorised rows."""
    M = np.array(M, copy=True)
    N = M.shape[0]
    inv = np.eye(N, dtype=M.dtype)
    for k in range(N):
        p = k + int(np.argmax(np.abs(M[k:, k])))
        if M[p, k] == 0:
            raise np.linalg.LinAlgError("singular")
        if p != k:
            M[[k, p]] = M[[p, k]]
            inv[[k, p]] = inv[[p, k]]
        d = M[k, k]
        M[k] = M[k] / d
        inv[k] = inv[k] / d
        col = M[:, k].copy()
        col[k] = 0
        M -= np.outer(col, M[k])
        inv -= np.outer(col, inv[k])
    return inv


def dense_green(A_diag, A_upper, A_lower, B_list=(), extended=False):
    """Selected blocks of G^R = A^-1 and of G^x = G^R B^x G^A for each B in B_list.

    B_list: sequence of (B_diag, B_upper) with B_lower = -B_upper^H.
    Returns dict(GR_full, GR=(diag,upper,lower), GX=[(diag,upper,lower), ...]).
    """
    n, b = A_diag.shape[0], A_diag.shape[1]
    dt = np.clongdouble if extended else np.complex128
    A = bt_to_dense(A_diag.astype(dt), A_upper.astype(dt), A_lower.astype(dt))
    GR = gauss_jordan_inverse(A) if extended else np.linalg.inv(A)
    out = {"GR_full": GR, "GR": dense_to_bt(GR, n, b), "GX": [], "GX_full": []}
    GA = dagger(GR)
    for (B_diag, B_upper) in B_list:
        B = bt_to_dense(B_diag.astype(dt), B_upper.astype(dt), -dagger(B_upper.astype(dt)))
        GX = GR @ B @ GA
        out["GX_full"].append(GX)
        out["GX"].append(dense_to_bt(GX, n, b))
    return out
