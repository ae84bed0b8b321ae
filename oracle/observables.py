"""Observables from the selected blocks (readings R11-R13).

TEST INFRASTRUCTURE (see oracle/__init__.py).  The paper shows local DOS (Fig. 4a,
PAPER.md:84, 94), spectral current and its conservation, transmission
(Fig. 6) and quotes an electron concentration; prefactors
(e/hbar, 2 pi, spin) are dropped as in R12-R13.
"""
import numpy as np

from .assemble import dagger


def ldos(GR_diag, GR_upper, GR_lower, S_diag=None, S_upper=None):
    """LDOS_i(E) = -(1/pi) Im Tr[(G^R S)_ii], (G^R S)_ii over the BT pattern (R12)."""
    n = GR_diag.shape[0]
    out = np.zeros(n)
    for i in range(n):
        if S_diag is None:
            tr = np.trace(GR_diag[i])
        else:
            tr = np.trace(GR_diag[i] @ S_diag[i])
            if i + 1 < n:
                tr += np.trace(GR_upper[i] @ dagger(S_upper[i]))      # G_{i,i+1} S_{i+1,i}
            if i > 0:
                tr += np.trace(GR_lower[i - 1] @ S_upper[i - 1])      # G_{i,i-1} S_{i-1,i}
        out[i] = -tr.imag / np.pi
    return out


def density_integrand(GL_diag, GL_upper, S_diag=None, S_upper=None):
    """Per-energy integrand Re[(-i/2pi) (G^< S)_kk] for k = 0..N-1 (R12); G^<_{i+1,i} = -(G^<_{i,i+1})^H."""
    n, b = GL_diag.shape[0], GL_diag.shape[1]
    out = np.zeros(n * b)
    for i in range(n):
        if S_diag is None:
            d = np.diagonal(GL_diag[i]).copy()
        else:
            d = np.einsum("kj,jk->k", GL_diag[i], S_diag[i])
            if i + 1 < n:
                d = d + np.einsum("kj,jk->k", GL_upper[i], dagger(S_upper[i]))
            if i > 0:
                d = d + np.einsum("kj,jk->k", -dagger(GL_upper[i - 1]), S_upper[i - 1])
        out[i * b:(i + 1) * b] = (-1j / (2 * np.pi) * d).real
    return out


def transmission(GR_corner0, gamma_L, gamma_R):
    """T(E) = Re Tr[Gamma_L G^R_{0,n-1} Gamma_R (G^R_{0,n-1})^H]  (R11)."""
    return float(np.trace(gamma_L @ GR_corner0 @ gamma_R @ dagger(GR_corner0)).real)


def bond_current(E, H_upper, S_upper, GL_upper):
    """J_i(E) = 2 Re Tr[(H_{i,i+1} - E S_{i,i+1}) G^<_{i+1,i}], G^<_{i+1,i} = -(G^<_{i,i+1})^H (R13)."""
    m = H_upper.shape[0]
    out = np.zeros(m)
    for i in range(m):
        hop = H_upper[i] if S_upper is None else H_upper[i] - E * S_upper[i]
        out[i] = 2.0 * np.trace(hop @ (-dagger(GL_upper[i]))).real
    return out


def contact_current(sig_l, sig_g, GL_block, GG_block):
    """Meir-Wingreen I(E) = Re Tr[Sigma^<_B G^> - Sigma^>_B G^<] on the contact block (R13)."""
    return float(np.trace(sig_l @ GG_block - sig_g @ GL_block).real)
