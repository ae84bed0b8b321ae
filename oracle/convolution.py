"""Eq. 3 of the paper: the energy convolution, by its definition.

TEST INFRASTRUCTURE (see oracle/__init__.py).  PAPER.md:60: B(E) ~ int dE' (M1 C1(E - E') M2) (.) C2(E'),
taken for M1 = M2 = I and (.) = element-wise product on the selected blocks (reading listed in
DESIGN.md section 2).  On a uniform grid of N_E energies, with zero outside the grid:
    convolution  Y[m] = scale * sum_k X1[m - k] * op(X2[k]),                 m = 0 .. 2 N_E - 2
    correlation  Y[m] = scale * sum_k X1[k] * op(X2[k - (m - (N_E - 1))])    (lag m - (N_E - 1))
op = identity or complex conjugate; optionally the b x b blocks of X2 transposed.  The sums are written
out as such (one vectorised product per pair of energies): no FFT here.
"""
import numpy as np


def _prepare_x2(X2, conj2, block):
    X2 = np.asarray(X2)
    if block:
        ne = X2.shape[0]
        X2 = np.swapaxes(X2.reshape(ne, -1, block, block), -1, -2).reshape(ne, -1)
    return np.conj(X2) if conj2 else X2


def energy_convolve(X1, X2, mode=0, conj2=False, scale=1.0, transpose_block=0):
    """X1, X2: [N_E, M] complex.  Returns Y [2 N_E - 1, M]."""
    X1 = np.asarray(X1)
    ne, M = X1.shape
    X2 = _prepare_x2(X2, conj2, transpose_block)
    Y = np.zeros((2 * ne - 1, M), dtype=np.complex128)
    for k1 in range(ne):
        for k2 in range(ne):
            m = k1 + k2 if mode == 0 else (k1 - k2) + (ne - 1)      # X1[k1] meets X2[k2]
            Y[m] += X1[k1] * X2[k2]
    return scale * Y
