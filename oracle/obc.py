"""Open-boundary self-energies by Sancho-Rubio decimation (doubling).

TEST INFRASTRUCTURE (see oracle/__init__.py).  The paper only says B "also contains an open
boundary condition term not shown here"; the algorithm is fixed by
BASELINE.json:north_star ("Sancho-Rubio decimation of the lead blocks") and written out in
SURVEY.md 8(c-2), followed here step by step on A-blocks (so S != I needs nothing extra).
"""
import numpy as np

from .assemble import dagger


def lead_blocks(z, H_d, H_u, S_d=None, S_u=None):
    """a_d = z S_d - H_d, a_u = z S_u - H_u, a_l = z S_u^H - H_u^H."""
    b = H_d.shape[0]
    Sd = np.eye(b) if S_d is None else S_d
    a_d = z * Sd - H_d
    if S_u is None:
        a_u = -H_u.astype(np.complex128)
        a_l = -dagger(H_u).astype(np.complex128)
    else:
        a_u = z * S_u - H_u
        a_l = z * dagger(S_u) - dagger(H_u)
    return a_d, a_u, a_l


def _inv(m):
    """LAPACK inverse in fp64; hand-written Gauss-Jordan (oracle/dense.py) in extended precision."""
    if m.dtype == np.clongdouble:
        from .dense import gauss_jordan_inverse
        return gauss_jordan_inverse(m)
    return np.linalg.inv(m)


def sancho_rubio(a_d, a_u, a_l, side, tol=1e-12, max_iter=64, extended=False, cond_trace=None):
    """Surface Green's function g_s of the semi-infinite lead.
    extended=True runs the SAME steps in 80-bit np.clongdouble (hazard H2: the fp64 doubling is
    conditioning-limited at ~eps/eta per step; the extended run is the yardstick for that).
    cond_trace: optional list that receives the 2-norm condition number of the inverted a_b of
    every doubling and of the final a_s (diagnostic for the H2 error bound; no effect on results).

    side 0 = left lead (surface cell couples rightwards into the device): a_s <- a_s - l g u
    side 1 = right lead:                                                  a_s <- a_s - u g l
    Each doubling: g = a_d^-1; a_s update; a_d <- a_d - u g l - l g u; u <- -u g u; l <- -l g l.
    Stop AFTER the update when ||u||_F + ||l||_F <= tol (||a_u||_F + ||a_l||_F) (reading R3).
    Returns (g_s, iters, converged)."""
    dt = np.clongdouble if extended else np.complex128
    a_s = a_d.astype(dt)
    a_b = a_d.astype(dt)
    u = a_u.astype(dt)
    l = a_l.astype(dt)
    ref = np.linalg.norm(a_u) + np.linalg.norm(a_l)
    iters, converged = 0, False
    for it in range(max_iter):
        if cond_trace is not None:
            cond_trace.append(float(np.linalg.cond(a_b.astype(np.complex128))))
        g = _inv(a_b)
        gu = g @ u
        gl = g @ l
        lgu = l @ gu
        ugl = u @ gl
        a_s = a_s - (lgu if side == 0 else ugl)
        a_b = a_b - ugl - lgu
        u = -(u @ gu)
        l = -(l @ gl)
        iters = it + 1
        if np.linalg.norm(u) + np.linalg.norm(l) <= tol * ref:
            converged = True
            break
    if cond_trace is not None:
        cond_trace.append(float(np.linalg.cond(a_s.astype(np.complex128))))
    return _inv(a_s), iters, converged


def boundary_self_energy(a_u, a_l, g_s, side):
    """Sigma^R_L = a_l g_s a_u (subtracted from A_00); Sigma^R_R = a_u g_s a_l (from A_{n-1,n-1})."""
    return a_l @ g_s @ a_u if side == 0 else a_u @ g_s @ a_l


def broadening(sigma_r):
    """Gamma = i (Sigma^R_B - Sigma^R_B^H)."""
    return 1j * (sigma_r - dagger(sigma_r))


def fermi(E, mu, kT):
    """f(E) = 1 / (1 + exp((E - mu)/kT)) at REAL E, overflow-safe."""
    x = (float(E) - mu) / kT
    if x > 0:
        ex = np.exp(-x)
        return ex / (1.0 + ex)
    return 1.0 / (1.0 + np.exp(x))


def boundary_lesser_greater(gamma, f):
    """Sigma^<_B = i f Gamma ; Sigma^>_B = -i (1 - f) Gamma."""
    return 1j * f * gamma, -1j * (1.0 - f) * gamma


def contact_blocks(H_diag, H_upper, S_diag, S_upper, side):
    """Reading R2: left lead = (H_00, S_00) with coupling (H_01, S_01);
    right lead = (H_{n-1,n-1}, S_{n-1,n-1}) with (H_{n-2,n-1}, S_{n-2,n-1})."""
    if side == 0:
        return (H_diag[0], H_upper[0], None if S_diag is None else S_diag[0],
                None if S_upper is None else S_upper[0])
    return (H_diag[-1], H_upper[-1], None if S_diag is None else S_diag[-1],
            None if S_upper is None else S_upper[-1])
