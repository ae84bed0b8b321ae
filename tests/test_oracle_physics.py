"""Physics pins for the whole oracle path (PAPER.md:86 current conservation).
CPU only."""
import numpy as np

from oracle import pipeline
from oracle.assemble import dagger
from paper_2602_03438_b200 import workloads as W


def _uniform_device(b, n, energies, eta=1e-7):
    H_d, H_u, U, eps, t = W.chain_lead(b)
    wl = W.make_workload(0, n_blocks=n, block_size=b, n_energy=len(energies))
    wl.H_diag = np.stack([H_d] * n)
    wl.H_upper = np.stack([H_u] * (n - 1))
    wl.energies = np.asarray(energies, float)
    wl.eta = eta
    wl.weights = W.trapezoid_weights(wl.energies)
    return wl, eps, t


def test_transmission_counts_open_channels():
    """P7: translation-invariant device => T(E) = #{k : |E - eps_k| < 2 t_k}; G_ii independent of i."""
    b, n = 5, 6
    energies = [-1.3, -0.4, 0.05, 0.6, 1.4, 2.5]
    wl, eps, t = _uniform_device(b, n, energies)
    for k, E in enumerate(energies):
        out = pipeline.solve_energy(wl, k)
        n_open = int(np.sum(np.abs(E - eps) < 2 * t))
        assert abs(out["obs"]["transmission"] - n_open) < 2e-4, (E, out["obs"]["transmission"], n_open)
        Gd = out["ret"]["GR_diag"]
        for i in range(1, n):
            assert np.linalg.norm(Gd[i] - Gd[0]) / np.linalg.norm(Gd[0]) < 1e-6
        # LDOS of a uniform chain is positive
        assert np.all(out["obs"]["ldos"] > 0)


def test_ballistic_current_conservation():
    """P8 (PAPER.md:86 'the electronic current remains perfectly conserved'):
    J_i(E) equal for all bonds, = I_L = -I_R = (f_L - f_R) T(E), up to O(eta)."""
    wl = W.make_workload(0, n_blocks=6, block_size=8, n_energy=5)
    wl.energies = np.linspace(-0.05, 0.25, 5)       # inside the bias window, f_L - f_R sizeable
    for k in range(5):
        out = pipeline.solve_energy(wl, k, want_greater=True)
        T = out["obs"]["transmission"]
        ref = (out["left"]["f"] - out["right"]["f"]) * T
        J = out["obs"]["bond_current"]
        I = out["obs"]["contact_current"]
        assert ref > 1e-4
        assert np.max(np.abs(J - ref)) < 2e-3 * ref
        assert abs(I[0] - ref) < 1e-6 * ref + 2e-3 * ref
        assert abs(I[1] + ref) < 2e-3 * ref


def test_equilibrium_fluctuation_dissipation():
    """P9: mu_L = mu_R, no Sigma_S => G^< = -f (G^R - G^A) up to the O(eta) term of hazard H1."""
    wl = W.make_workload(0, n_blocks=4, block_size=6, n_energy=1)
    wl.mu_L = wl.mu_R = 0.25
    wl.eta = 1e-9
    out = pipeline.solve_energy(wl, 0)
    f = out["left"]["f"]
    G = out["ret"]["GR_diag"]
    ref = -f * (G - dagger(G))
    err = np.linalg.norm(out["les"]["GX_diag"] - ref) / np.linalg.norm(ref)
    assert err < 1e-5
    # then density integrand_k = -(f/pi) Im G_kk, i.e. sum_k = f * sum_i LDOS_i
    dens = out["obs"]["density_integrand"]
    assert np.all(dens > -1e-12)
    assert abs(dens.sum() - f * out["obs"]["ldos"].sum()) < 1e-5 * abs(dens.sum())


def test_density_uses_overlap_pattern():
    """R12: with S != I the density needs the off-diagonal blocks: compare against the dense
    diag(G^< S)."""
    from oracle import assemble, dense
    wl = W.make_workload(2, n_blocks=4, block_size=5, n_energy=2)
    out = pipeline.solve_energy(wl, 1)
    d = dense.dense_green(*out["A"], B_list=[out["BL"]])
    S = assemble.bt_to_dense(wl.S_diag, wl.S_upper, dagger(wl.S_upper))
    ref = (-1j / (2 * np.pi) * np.diagonal(d["GX_full"][0] @ S)).real
    assert np.allclose(out["obs"]["density_integrand"], ref, rtol=1e-9, atol=1e-14)
    GS = d["GR_full"] @ S
    b = wl.block_size
    ref_ldos = np.array([-np.trace(GS[i * b:(i + 1) * b, i * b:(i + 1) * b]).imag / np.pi for i in range(4)])
    assert np.allclose(out["obs"]["ldos"], ref_ldos, rtol=1e-9)
