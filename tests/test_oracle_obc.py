"""Pins for oracle/obc.py.  CPU only."""
import numpy as np
import pytest

from oracle import obc
from oracle.assemble import dagger
from paper_2602_03438_b200 import workloads as W


def chain_surface_gf(z, eps, t):
    """Closed form for the semi-infinite 1D chain, on-site eps, hopping -t (P5):
    g = [(z-eps) - sqrt((z-eps)^2 - 4 t^2)] / (2 t^2), retarded branch Im g < 0."""
    w = z - eps
    s = np.sqrt(w * w - 4 * t * t + 0j)
    g1, g2 = (w - s) / (2 * t * t), (w + s) / (2 * t * t)
    return g1 if g1.imag < 0 else g2


@pytest.mark.parametrize("E", [-2.5, -1.99, -0.7, 0.013, 0.3, 1.2, 2.0, 2.7])
@pytest.mark.parametrize("side", [0, 1])
def test_1d_chain_closed_form(E, side):
    """Inside (|E|<2t), at the edge of, and outside the band; t = 1, eps = 0.
    E = 0 exactly is avoided: every odd-length isolated segment has an eigenvalue exactly there,
    so g = a_d^-1 ~ 1/eta and the doubling loses ~5 digits (hazard H2 in its extreme form;
    test_chain_band_centre_is_conditioning_limited records it)."""
    eta = 1e-6
    z = complex(E, eta)
    a_d, a_u, a_l = obc.lead_blocks(z, np.array([[0.0 + 0j]]), np.array([[-1.0 + 0j]]))
    g, iters, conv = obc.sancho_rubio(a_d, a_u, a_l, side, 1e-12, 64)
    ref = chain_surface_gf(z, 0.0, 1.0)
    assert conv and iters < 40
    assert abs(g[0, 0] - ref) < 2e-8 * abs(ref)      # conditioning-limited near band edges (H2)
    sig = obc.boundary_self_energy(a_u, a_l, g, side)
    assert abs(sig[0, 0] - ref) < 2e-8 * abs(ref)     # Sigma = t^2 g, t = 1


@pytest.mark.parametrize("b", [3, 8])
def test_unitary_mixed_chains(b):
    """P5 for any b: H_d = U diag(eps) U^H, H_u = U diag(-t) U^H => g_s = U diag(g_k) U^H."""
    H_d, H_u, U, eps, t = W.chain_lead(b)
    eta = 1e-5
    for E in (-0.9, 0.1, 0.45, 1.7):
        z = complex(E, eta)
        a_d, a_u, a_l = obc.lead_blocks(z, H_d, H_u)
        gk = np.array([chain_surface_gf(z, eps[k], t[k]) for k in range(b)])
        ref = (U * gk) @ U.conj().T
        for side in (0, 1):
            g, iters, conv = obc.sancho_rubio(a_d, a_u, a_l, side, 1e-12, 64)
            assert conv
            assert np.linalg.norm(g - ref) / np.linalg.norm(ref) < 1e-8
            sig = obc.boundary_self_energy(a_u, a_l, g, side)
            sig_ref = (U * (t * t * gk)) @ U.conj().T
            assert np.linalg.norm(sig - sig_ref) / np.linalg.norm(sig_ref) < 1e-8


def test_left_right_differ_and_fixed_point():
    """P6 (necessary): g_L = (a_d - a_l g_L a_u)^-1 and g_R = (a_d - a_u g_R a_l)^-1; a
    non-symmetric lead distinguishes the two sides (catches a swapped side)."""
    wl = W.make_workload(2, n_blocks=3, block_size=6, n_energy=1)
    z = complex(0.3, 1e-4)
    for side in (0, 1):
        Hd, Hu, Sd, Su = obc.contact_blocks(wl.H_diag, wl.H_upper, wl.S_diag, wl.S_upper, side)
        a_d, a_u, a_l = obc.lead_blocks(z, Hd, Hu, Sd, Su)
        g, iters, conv = obc.sancho_rubio(a_d, a_u, a_l, side)
        assert conv
        if side == 0:
            fp = np.linalg.inv(a_d - a_l @ g @ a_u)
            wrong = np.linalg.inv(a_d - a_u @ g @ a_l)
        else:
            fp = np.linalg.inv(a_d - a_u @ g @ a_l)
            wrong = np.linalg.inv(a_d - a_l @ g @ a_u)
        assert np.linalg.norm(fp - g) / np.linalg.norm(g) < 1e-8
        assert np.linalg.norm(wrong - g) / np.linalg.norm(g) > 1e-3


def test_retarded_sign_and_gamma_psd():
    """Gamma = i(Sigma - Sigma^H) is Hermitian positive semi-definite for a retarded Sigma."""
    wl = W.make_workload(0)
    from oracle import pipeline
    for side, mu in ((0, wl.mu_L), (1, wl.mu_R)):
        o = pipeline.obc_one_energy(0.3, wl.eta, wl.H_diag, wl.H_upper, None, None, mu, wl.kT, side)
        gam = o["gamma"]
        assert np.abs(gam - dagger(gam)).max() < 1e-12
        assert np.linalg.eigvalsh(gam).min() > -1e-9
        assert np.allclose(o["sigma_l"], 1j * o["f"] * gam)
        assert np.allclose(o["sigma_g"] - o["sigma_l"], o["sigma_r"] - dagger(o["sigma_r"]))


def test_fermi_overflow_safe():
    assert obc.fermi(1e4, 0.0, 0.025) == 0.0
    assert obc.fermi(-1e4, 0.0, 0.025) == 1.0
    assert abs(obc.fermi(0.1, 0.1, 0.025) - 0.5) < 1e-15
    assert abs(obc.fermi(0.125, 0.1, 0.025) - 1 / (1 + np.e)) < 1e-15


def test_max_iter_reported():
    a_d, a_u, a_l = obc.lead_blocks(complex(0.0, 1e-6), np.array([[0.0 + 0j]]), np.array([[-1.0 + 0j]]))
    g, iters, conv = obc.sancho_rubio(a_d, a_u, a_l, 0, 1e-12, 5)
    assert iters == 5 and not conv


def test_chain_band_centre_is_conditioning_limited():
    """Hazard H2, extreme case: at E = eps exactly the algorithm itself (not the oracle's coding)
    is accurate only to ~eps_machine/eta-amplified level; it must still converge and land within 1e-3."""
    z = complex(0.0, 1e-6)
    a_d, a_u, a_l = obc.lead_blocks(z, np.array([[0.0 + 0j]]), np.array([[-1.0 + 0j]]))
    g, iters, conv = obc.sancho_rubio(a_d, a_u, a_l, 0, 1e-12, 64)
    assert conv
    assert abs(g[0, 0] - chain_surface_gf(z, 0.0, 1.0)) < 1e-3


def test_extended_precision_decimation_is_the_yardstick():
    """The 80-bit run of the same doubling reproduces the 1D closed form far better than fp64 where
    fp64 is conditioning-limited (H2), which justifies using it to judge decimation parity."""
    z = complex(0.013, 1e-6)
    a_d, a_u, a_l = obc.lead_blocks(z, np.array([[0.0 + 0j]]), np.array([[-1.0 + 0j]]))
    ref = chain_surface_gf(z, 0.0, 1.0)
    g64, _, c64 = obc.sancho_rubio(a_d, a_u, a_l, 0)
    g80, _, c80 = obc.sancho_rubio(a_d, a_u, a_l, 0, extended=True)
    assert c64 and c80 and g80.dtype == np.clongdouble
    e64, e80 = abs(g64[0, 0] - ref), abs(complex(g80[0, 0]) - ref)
    assert e80 < 1e-12 and e80 <= e64
    # and on a matrix lead: unitary-mixed chains
    H_d, H_u, U, eps, t = W.chain_lead(6)
    z = complex(0.1, 1e-6)
    a_d, a_u, a_l = obc.lead_blocks(z, H_d, H_u)
    gk = np.array([chain_surface_gf(z, eps[k], t[k]) for k in range(6)])
    refm = (U * gk) @ U.conj().T
    g80, _, _ = obc.sancho_rubio(a_d, a_u, a_l, 1, extended=True)
    assert np.linalg.norm(g80.astype(np.complex128) - refm) / np.linalg.norm(refm) < 1e-11
