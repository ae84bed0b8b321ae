"""The same Eqs. 1-2 for the other populations of the paper (C = D or W, A made of the
dynamical or bare Coulomb matrix), as mappings onto the inputs of the electron
path.  These pins check the oracle under each mapping against something that is not the oracle:
the Bloch-mode count of a perfect phonon wire and the Dyson equation of the screened interaction
solved as one dense linear system."""
import numpy as np

from oracle import assemble, pipeline
from paper_2602_03438_b200 import workloads as W


def _bloch_mode_count(Phi_d, Phi_u, w2, nk=4001):
    """Number of right-moving Bloch modes of the wire at omega^2 = w2: crossings of the bands
    lambda_j(k) of Phi(k) = Phi_d + Phi_u e^{ik} + Phi_u^H e^{-ik} with w2 for k in (0, pi)."""
    ks = np.linspace(0.0, np.pi, nk)
    bands = np.array([np.linalg.eigvalsh(Phi_d + Phi_u * np.exp(1j * k) + Phi_u.conj().T * np.exp(-1j * k)) for k in ks])
    s = np.sign(bands - w2)
    return int(np.sum(s[1:] * s[:-1] < 0))


def test_phonon_wire_inputs_obey_the_acoustic_sum_rule():
    wl = W.make_phonon_workload(6, 4, 3, periodic=True)
    cell = wl.H_diag[2] + wl.H_upper[2] + wl.H_upper[1].conj().T
    assert np.abs(cell.sum(axis=1)).max() < 1e-14          # a rigid translation costs no energy
    assert np.allclose(wl.H_diag[0], wl.H_diag[3]) and np.allclose(wl.H_diag[5], wl.H_diag[3])
    assert np.linalg.eigvalsh(wl.H_diag[0]).min() > 0 and np.all(wl.energies > 0)


def test_phonon_wire_transmission_counts_bloch_modes():
    """A perfect wire transmits one quantum per propagating mode: T(w) = number of Bloch bands crossing
    w^2 (Landauer); the decimation, the sweeps and the Caroli trace all enter."""
    wl = W.make_phonon_workload(4, 5, 6, periodic=True, eta=1e-9)
    wl.energies = np.array([0.4, 1.0, 1.8, 1.9, 2.0, 2.6])      # acoustic branch alone, optical branches, upper band
    seen = set()
    for k in range(wl.n_energy):
        w2 = float(wl.energies[k])
        modes = _bloch_mode_count(wl.H_diag[1], wl.H_upper[1], w2)
        out = pipeline.solve_energy(wl, k, want_greater=False)
        assert out["left"]["converged"] and out["right"]["converged"]
        assert abs(out["obs"]["transmission"] - modes) < 1e-5, (w2, modes, out["obs"]["transmission"])
        seen.add(modes)
    assert len(seen) > 1 and max(seen) >= 2      # the grid crosses band edges: more than one plateau


def test_coulomb_mapping_solves_the_dyson_equation():
    """H := -V^-1, z = 0, Sigma := P  gives  W^R = (V^-1 - P^R)^-1 = (I - V P^R)^-1 V  and
    W^<> = W^R P^<> W^A: checked against ONE dense solve with V itself."""
    wl, sig = W.make_coulomb_workload(4, 6, 2)
    n, b = wl.n_blocks, wl.block_size
    Vinv = assemble.bt_to_dense(-wl.H_diag, -wl.H_upper, -np.conj(np.swapaxes(wl.H_upper, -1, -2)))
    V = np.linalg.inv(Vinv)
    zero = {k: np.zeros((b, b), complex) for k in ("sigma_r", "gamma", "sigma_l", "sigma_g")}
    h = lambda a: np.conj(np.swapaxes(a, -1, -2))
    for k in range(wl.n_energy):
        s1 = {t: {kk: (vv[k:k + 1] if kk != "kind" else vv) for kk, vv in sig[t].items()} for t in "rlg"}
        out = pipeline.solve_energy(wl, k, sigma=s1, obc_in=(zero, zero), want_greater=True, corner=False)
        PR = assemble.bt_to_dense(sig["r"]["diag"][k], sig["r"]["upper"][k], sig["r"]["lower"][k])
        WR = np.linalg.solve(np.eye(n * b) - V @ PR, V)
        d, u, l = assemble.dense_to_bt(WR, n, b)
        assert np.abs(out["ret"]["GR_diag"] - d).max() < 1e-11 * np.abs(d).max()
        assert np.abs(out["ret"]["GR_upper"] - u).max() < 1e-11 * np.abs(d).max()
        assert np.abs(out["ret"]["GR_lower"] - l).max() < 1e-11 * np.abs(d).max()
        for t, grp in (("l", "les"), ("g", "gtr")):
            PX = assemble.bt_to_dense(sig[t]["diag"][k], sig[t]["upper"][k], -h(sig[t]["upper"][k]))
            WX = WR @ PX @ WR.conj().T
            dx, ux, _ = assemble.dense_to_bt(WX, n, b)
            assert np.abs(out[grp]["GX_diag"] - dx).max() < 1e-11 * np.abs(dx).max()
            assert np.abs(out[grp]["GX_upper"] - ux).max() < 1e-11 * np.abs(dx).max()
