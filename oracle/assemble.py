"""Assembly of the block-tridiagonal A(E) = z S - H - Sigma^R and B^<> = Sigma^<>.

TEST INFRASTRUCTURE (see oracle/__init__.py).  Follows PAPER.md:56 (Eq. 1: C^R = (A - B^R)^-1
with A = E S - H for electrons) and SURVEY.md 8(a) row S1.
z = E + i*eta multiplies S everywhere (reading R1).
"""
import numpy as np


def dagger(a):
    return np.conj(np.swapaxes(a, -1, -2))


def a_blocks(z, H_diag, H_upper, S_diag=None, S_upper=None, sigma_r=None,
             sigma_left=None, sigma_right=None):
    """Blocks of A = z S - H - Sigma^R_S - Sigma^R_B for ONE energy.

    H_diag [n,b,b], H_upper [n-1,b,b] (H_lower = H_upper^H, H Hermitian).
    S_* None => S = I.  sigma_r: None | {"kind":"scalar","value":s} (s*I on every
    diagonal block) | {"kind":"bt","diag","upper","lower"} for this energy.
    sigma_left/right: boundary self-energies subtracted from blocks 0 and n-1.
    Returns (A_diag [n,b,b], A_upper [n-1,b,b], A_lower [n-1,b,b]).
    NOTE A_lower[i] = A_{i+1,i} = z S_{i,i+1}^H - H_{i,i+1}^H - Sigma_{i+1,i}; z is NOT conjugated.
    """
    n, b = H_diag.shape[0], H_diag.shape[1]
    eye = np.eye(b)
    A_diag = np.empty((n, b, b), dtype=np.result_type(H_diag.dtype, np.complex128))
    A_upper = np.empty((max(n - 1, 0), b, b), dtype=A_diag.dtype)
    A_lower = np.empty_like(A_upper)
    for i in range(n):
        Sii = eye if S_diag is None else S_diag[i]
        A_diag[i] = z * Sii - H_diag[i]
    for i in range(n - 1):
        if S_upper is None:
            A_upper[i] = -H_upper[i]
            A_lower[i] = -dagger(H_upper[i])
        else:
            A_upper[i] = z * S_upper[i] - H_upper[i]
            A_lower[i] = z * dagger(S_upper[i]) - dagger(H_upper[i])
    if sigma_r is not None:
        if sigma_r["kind"] == "scalar":
            for i in range(n):
                A_diag[i] -= sigma_r["value"] * eye
        else:
            A_diag -= sigma_r["diag"]
            A_upper -= sigma_r["upper"]
            A_lower -= sigma_r["lower"]
    if sigma_left is not None:
        A_diag[0] -= sigma_left
    if sigma_right is not None:
        A_diag[n - 1] -= sigma_right
    return A_diag, A_upper, A_lower


def b_blocks(n, b, sigma_x=None, sigma_left=None, sigma_right=None, dtype=np.complex128):
    """Blocks of B^<> = Sigma^<>_S + Sigma^<>_B for ONE energy (Eq. 2 right side).
    Returns (B_diag [n,b,b], B_upper [n-1,b,b]); B_lower = -B_upper^H (anti-Hermitian B)."""
    B_diag = np.zeros((n, b, b), dtype=dtype)
    B_upper = np.zeros((max(n - 1, 0), b, b), dtype=dtype)
    if sigma_x is not None:
        if sigma_x["kind"] == "scalar":
            for i in range(n):
                B_diag[i] += sigma_x["value"] * np.eye(b)
        else:
            B_diag += sigma_x["diag"]
            B_upper += sigma_x["upper"]
    if sigma_left is not None:
        B_diag[0] += sigma_left
    if sigma_right is not None:
        B_diag[n - 1] += sigma_right
    return B_diag, B_upper


def bt_to_dense(diag, upper, lower):
    """Full N x N matrix from BT blocks (tier-0 helper)."""
    n, b = diag.shape[0], diag.shape[1]
    M = np.zeros((n * b, n * b), dtype=diag.dtype)
    for i in range(n):
        M[i * b:(i + 1) * b, i * b:(i + 1) * b] = diag[i]
    for i in range(n - 1):
        M[i * b:(i + 1) * b, (i + 1) * b:(i + 2) * b] = upper[i]
        M[(i + 1) * b:(i + 2) * b, i * b:(i + 1) * b] = lower[i]
    return M


def dense_to_bt(M, n, b):
    """Selected blocks (i,i), (i,i+1), (i+1,i) of a dense matrix."""
    diag = np.stack([M[i * b:(i + 1) * b, i * b:(i + 1) * b] for i in range(n)])
    if n > 1:
        upper = np.stack([M[i * b:(i + 1) * b, (i + 1) * b:(i + 2) * b] for i in range(n - 1)])
        lower = np.stack([M[(i + 1) * b:(i + 2) * b, i * b:(i + 1) * b] for i in range(n - 1)])
    else:
        upper = np.zeros((0, b, b), M.dtype)
        lower = np.zeros((0, b, b), M.dtype)
    return diag, upper, lower
