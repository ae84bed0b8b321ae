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


def _overlap_chain_device(b, n, energies, eta, seed=11):
    """Translation-invariant device WITH overlap whose modes decouple in one unitary basis U:
    H_d = U diag(eps) U^H, H_u = U diag(h) U^H, S_d = U diag(1 + s) U^H, S_u = U diag(sig) U^H with COMPLEX
    h_k and sig_k, so that S_u and H_u are not Hermitian (S_u^H != S_u) and every mode k is a 1D chain with
    a_d = z (1 + s_k) - eps_k, a_u = z sig_k - h_k, a_l = z conj(sig_k) - conj(h_k)   (z NOT conjugated).
    Input construction only; the closed forms are in the tests."""
    _, _, U, eps, t = W.chain_lead(b)
    rng = np.random.default_rng(seed)
    h = -t * np.exp(1j * rng.uniform(-1.0, 1.0, b))
    s = rng.uniform(-0.1, 0.1, b)
    sig = 0.08 * rng.uniform(0.5, 1.0, b) * np.exp(1j * rng.uniform(-np.pi, np.pi, b))
    mk = lambda d: (U * d) @ U.conj().T
    wl = W.make_workload(2, n_blocks=n, block_size=b, n_energy=len(energies))
    wl.H_diag, wl.H_upper = np.stack([mk(eps)] * n), np.stack([mk(h)] * (n - 1))
    wl.S_diag, wl.S_upper = np.stack([mk(1 + s)] * n), np.stack([mk(sig)] * (n - 1))
    wl.energies = np.asarray(energies, float)
    wl.eta = eta
    wl.weights = W.trapezoid_weights(wl.energies)
    return wl, U, eps, h, s, sig


def test_overlap_chain_bulk_green_function_closed_form():
    """Pins assemble.a_blocks with S != I (A_upper = z S_u - H_u, A_lower = z S_u^H - H_u^H, z not conjugated):
    in the mode basis the infinite chain has G_ii = U diag(1 / sqrt(a_d^2 - 4 a_u a_l)) U^H for every i
    (root with a_d - 2 a_u a_l g_s, g_s the decaying surface solution).  eta is LARGE here (0.05) so that
    conj(z) in place of z, a dropped dagger on S_u or H_u, or a wrong sign each move the result by percents."""
    b, n, eta = 5, 5, 0.05
    energies = [-0.8, -0.2, 0.1, 0.55, 1.3]
    wl, U, eps, h, s, sig = _overlap_chain_device(b, n, energies, eta)
    for k, E in enumerate(energies):
        z = complex(E, eta)
        a_d = z * (1 + s) - eps
        a_u = z * sig - h
        a_l = z * np.conj(sig) - np.conj(h)
        root = np.sqrt(a_d * a_d - 4 * a_u * a_l + 0j)
        g1, g2 = (a_d - root) / (2 * a_u * a_l), (a_d + root) / (2 * a_u * a_l)
        gs = np.where(np.abs(g1 * g1 * a_u * a_l) < 1, g1, g2)         # decaying solution
        Gk = 1.0 / (a_d - 2 * a_u * a_l * gs)
        ref = (U * Gk) @ U.conj().T
        out = pipeline.solve_energy(wl, k)
        Gd = out["ret"]["GR_diag"]
        for i in range(n):
            assert np.linalg.norm(Gd[i] - ref) / np.linalg.norm(ref) < 1e-9, (E, i)
        # first off-diagonal blocks of the infinite chain: G_{i,i+1} = -g_s a_u G_{i+1,i+1}, G_{i+1,i} = -g_s a_l G_ii
        up = (U * (-gs * a_u * Gk)) @ U.conj().T
        lo = (U * (-gs * a_l * Gk)) @ U.conj().T
        assert np.linalg.norm(out["ret"]["GR_upper"][1] - up) / np.linalg.norm(up) < 1e-9
        assert np.linalg.norm(out["ret"]["GR_lower"][2] - lo) / np.linalg.norm(lo) < 1e-9


def test_overlap_chain_transmission_counts_open_channels():
    """P7 with S != I: T(E) = #{k : |a_d,k(E)| < 2 |a_u,k(E)|} at real E (generalised bands), G_ii independent of i."""
    b, n = 5, 6
    energies = [-1.1, -0.35, 0.07, 0.5, 1.25, 2.4]
    wl, U, eps, h, s, sig = _overlap_chain_device(b, n, energies, 1e-7)
    seen = set()
    for k, E in enumerate(energies):
        n_open = int(np.sum(np.abs(E * (1 + s) - eps) < 2 * np.abs(E * sig - h)))
        seen.add(n_open)
        out = pipeline.solve_energy(wl, k)
        assert abs(out["obs"]["transmission"] - n_open) < 5e-4, (E, out["obs"]["transmission"], n_open)
        Gd = out["ret"]["GR_diag"]
        for i in range(1, n):
            assert np.linalg.norm(Gd[i] - Gd[0]) / np.linalg.norm(Gd[0]) < 1e-5
    assert len(seen) >= 3           # the grid really crosses band edges


def test_ballistic_current_conservation_with_overlap():
    """P8 on a configs[2]-shaped device (non-orthogonal S, no Sigma_S): every bond current
    J_i = 2 Re Tr[(H_{i,i+1} - E S_{i,i+1}) G^<_{i+1,i}] equals I_L = -I_R = (f_L - f_R) T(E) up to O(eta).
    Dropping or mis-signing the E S_{i,i+1} term of observables.bond_current breaks it at the percent level
    (checked below by doing exactly that to a copy of the formula's input)."""
    from oracle import observables
    wl = W.make_workload(2, n_blocks=5, block_size=8, n_energy=6)
    wl.S_upper = wl.S_upper * 6.0                    # overlap coupling comparable to H_upper x |E|: the term matters
    wl.energies = np.array([-1.0, -0.9, -0.2, 0.2, 0.9, 1.0])      # energies where this small device conducts
    wl.eta = 1e-8                                    # conservation holds up to O(eta)
    wl.mu_L, wl.mu_R, wl.kT = 0.9, -0.9, 0.2         # wide bias window: f_L - f_R sizeable at every energy
    sens = 1e9
    for k in range(6):
        out = pipeline.solve_energy(wl, k, want_greater=True)
        T = out["obs"]["transmission"]
        ref = (out["left"]["f"] - out["right"]["f"]) * T
        J = out["obs"]["bond_current"]
        I = out["obs"]["contact_current"]
        assert ref > 5e-2
        assert np.max(np.abs(J - ref)) < 2e-5 * ref, (k, J, ref)
        assert abs(I[0] - ref) < 2e-6 * ref and abs(I[1] + ref) < 2e-6 * ref
        wrong = observables.bond_current(float(wl.energies[k]), wl.H_upper, None, out["les"]["GX_upper"])
        sens = min(sens, float(np.max(np.abs(wrong - ref)) / ref))
    assert sens > 0.1               # without the overlap term the currents are NOT conserved, at every energy
