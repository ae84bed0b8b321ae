"""Tier 1 - recursive Green's function (RGF) sweeps, block by block.

TEST INFRASTRUCTURE (see oracle/__init__.py).  "Eqs. (1) and (2) can be solved with the
so-called recursive Green's function (RGF) algorithm, which is sequential in essence [10]"
(PAPER.md:72).  The paper prints no recurrences; these are SURVEY.md 8(a) rows S3-S6 and
8(c-1), i.e. block Gaussian elimination of Eqs. 1-2, in that order and notation:
  g_i    left-connected retarded GF,  X_i = g_i A_{i,i+1},  Y_i = A_{i+1,i} g_i
  g^x_i  left-connected lesser/greater GF.
Daggers are daggers of A's OWN blocks (A is not Hermitian): A_{i,i-1}^H is never A_{i-1,i}.
One np.linalg.inv and plain @ products per step; no blocking, fusion or reordering.
"""
import numpy as np

from .assemble import dagger


def rgf_retarded(A_diag, A_upper, A_lower, corner=False):
    """S3 (forward) + S4 (backward).  Returns dict with
    GR_diag [n,b,b], GR_upper [n-1] (G_{i,i+1}), GR_lower [n-1] (G_{i+1,i}),
    GR_corner ([n,b,b] column G_{i,n-1}, if corner), and the sweep state g, X, Y."""
    n, b = A_diag.shape[0], A_diag.shape[1]
    dt = A_diag.dtype
    g = np.empty((n, b, b), dt)
    X = np.empty((max(n - 1, 0), b, b), dt)   # X_i = g_i A_{i,i+1}
    Y = np.empty((max(n - 1, 0), b, b), dt)   # Y_i = A_{i+1,i} g_i
    # S3: g_0 = A_00^-1 ; g_i = (A_ii - A_{i,i-1} g_{i-1} A_{i-1,i})^-1
    g[0] = np.linalg.inv(A_diag[0])
    for i in range(1, n):
        Y[i - 1] = A_lower[i - 1] @ g[i - 1]
        g[i] = np.linalg.inv(A_diag[i] - Y[i - 1] @ A_upper[i - 1])
    # S4
    GR_diag = np.empty_like(g)
    GR_upper = np.empty_like(X)
    GR_lower = np.empty_like(X)
    GR_diag[n - 1] = g[n - 1]
    col = None
    if corner:
        col = np.empty_like(g)
        col[n - 1] = g[n - 1]
    for i in range(n - 2, -1, -1):
        X[i] = g[i] @ A_upper[i]
        GR_upper[i] = -X[i] @ GR_diag[i + 1]
        GR_lower[i] = -GR_diag[i + 1] @ Y[i]
        GR_diag[i] = g[i] - GR_upper[i] @ Y[i]
        if corner:
            col[i] = -X[i] @ col[i + 1]          # G_{i,n-1} = -X_i G_{i+1,n-1}
    return {"GR_diag": GR_diag, "GR_upper": GR_upper, "GR_lower": GR_lower,
            "GR_corner": col, "g": g, "X": X, "Y": Y}


def rgf_lesser_greater(A_upper, A_lower, B_diag, B_upper, ret):
    """S5 (forward) + S6 (backward) for ONE of </>; B = Sigma^x (B_lower = -B_upper^H).
    `ret` is the dict returned by rgf_retarded for the same A.
    Returns dict GX_diag [n,b,b], GX_upper [n-1] (G^x_{i,i+1}), GX_lower [n-1] = -GX_upper^H,
    plus gx (left-connected)."""
    g, X, Y, GR_diag = ret["g"], ret["X"], ret["Y"], ret["GR_diag"]
    n, b = g.shape[0], g.shape[1]
    gx = np.empty_like(g)
    # S5: g^x_0 = g_0 B_00 g_0^H
    gx[0] = g[0] @ B_diag[0] @ dagger(g[0])
    for i in range(1, n):
        Al = A_lower[i - 1]                     # A_{i,i-1}
        B_low = -dagger(B_upper[i - 1])         # B_{i,i-1}
        inner = (B_diag[i] + Al @ gx[i - 1] @ dagger(Al)
                 - Y[i - 1] @ B_upper[i - 1] - B_low @ dagger(Y[i - 1]))
        gx[i] = g[i] @ inner @ dagger(g[i])
    # S6
    GX_diag = np.empty_like(g)
    GX_upper = np.empty_like(X)
    GX_lower = np.empty_like(X)
    GX_diag[n - 1] = gx[n - 1]
    for i in range(n - 2, -1, -1):
        GX_upper[i] = ((-gx[i] @ dagger(A_lower[i]) + g[i] @ B_upper[i]) @ dagger(GR_diag[i + 1])
                       - X[i] @ GX_diag[i + 1])
        GX_lower[i] = -dagger(GX_upper[i])
        GX_diag[i] = (gx[i] - X[i] @ GX_lower[i] - GX_upper[i] @ dagger(X[i])
                      - X[i] @ GX_diag[i + 1] @ dagger(X[i]))
    return {"GX_diag": GX_diag, "GX_upper": GX_upper, "GX_lower": GX_lower, "gx": gx}


def lower_block_independent(A_upper, A_lower, B_upper, ret, les, i):
    """Cross-check of SURVEY.md 8(c-1): G^x_{i+1,i} computed WITHOUT using anti-Hermiticity,
      G^x_{i+1,i} = -G^R_{i+1,i+1} A_{i+1,i} g^x_i + G^R_{i+1,i+1} B_{i+1,i} g_i^H
                    - G^x_{i+1,i+1} A_{i,i+1}^H g_i^H."""
    g, GR = ret["g"], ret["GR_diag"]
    B_low = -dagger(B_upper[i])
    return (-GR[i + 1] @ A_lower[i] @ les["gx"][i] + GR[i + 1] @ B_low @ dagger(g[i])
            - les["GX_diag"][i + 1] @ dagger(A_upper[i]) @ dagger(g[i]))


def diag_block_six_terms(A_upper, A_lower, B_upper, ret, les, i):
    """Cross-check of SURVEY.md 8(c-1): fully expanded six-term form of G^x_ii."""
    g, GR = ret["g"], ret["GR_diag"]
    Xi = g[i] @ A_upper[i]
    G = GR[i + 1]
    gx = les["gx"][i]
    B_up = B_upper[i]
    B_low = -dagger(B_upper[i])
    Al = A_lower[i]
    return (gx + Xi @ les["GX_diag"][i + 1] @ dagger(Xi)
            + gx @ dagger(Al) @ dagger(G) @ dagger(Xi) + Xi @ G @ Al @ gx
            - g[i] @ B_up @ dagger(G) @ dagger(Xi) - Xi @ G @ B_low @ dagger(g[i]))
