"""The seeded generator: determinism, structure, distributions (readings R4-R10).  CPU only."""
import numpy as np

from paper_2602_03438_b200 import workloads as W


def test_deterministic_and_shapes():
    a = W.make_workload(1, n_blocks=4, block_size=8, n_energy=5)
    b = W.make_workload(1, n_blocks=4, block_size=8, n_energy=5)
    assert np.array_equal(a.H_diag, b.H_diag) and np.array_equal(a.H_upper, b.H_upper)
    assert a.H_diag.shape == (4, 8, 8) and a.H_upper.shape == (3, 8, 8)
    assert a.energies[0] == -1.0 and a.energies[-1] == 1.0
    assert abs(a.weights.sum() - 2.0) < 1e-14
    w0 = W.make_workload(0)
    assert w0.energies.tolist() == [0.3] and w0.eta == 1e-6 and (w0.n_blocks, w0.block_size) == (8, 16)


def test_hermitian_and_variances():
    wl = W.make_workload(0, n_blocks=6, block_size=64)
    Hd = wl.H_diag
    assert np.abs(Hd - np.conj(np.swapaxes(Hd, -1, -2))).max() == 0.0
    b = 64
    off = Hd[:, ~np.eye(b, dtype=bool)]
    assert abs(np.mean(np.abs(off) ** 2) * b - 1.0) < 0.05          # CN(0,1)/sqrt(b)
    assert abs(np.mean(np.abs(wl.H_upper) ** 2) * b - 0.5) < 0.03   # CN(0,0.5)/sqrt(b)
    w2 = W.make_workload(2, n_blocks=3, block_size=32, n_energy=2)
    assert abs(np.mean(np.abs(w2.H_upper) ** 2) * 32 - 0.5 * 0.49) < 0.03
    assert np.abs(w2.S_diag - np.conj(np.swapaxes(w2.S_diag, -1, -2))).max() == 0.0
    assert np.linalg.eigvalsh(w2.S_diag[0]).min() > 0.5


def test_bt_sigma_identity():
    """R6: Sigma^> - Sigma^< = Sigma^R - Sigma^A as full matrices; Sigma^<> anti-Hermitian."""
    wl = W.make_workload(3, n_blocks=3, block_size=4, n_energy=2)
    s = wl.sigma_s(0, 2)
    h = lambda a: np.conj(np.swapaxes(a, -1, -2))
    for k in range(2):
        assert np.allclose(s["g"]["diag"][k] - s["l"]["diag"][k], s["r"]["diag"][k] - h(s["r"]["diag"][k]))
        assert np.allclose(s["g"]["upper"][k] - s["l"]["upper"][k], s["r"]["upper"][k] - h(s["r"]["lower"][k]))
        assert np.allclose(s["l"]["diag"][k], -h(s["l"]["diag"][k]))
    # per-energy streams: a sub-range reproduces the same arrays
    s1 = wl.sigma_s(1, 2)
    assert np.array_equal(s1["r"]["diag"][0], s["r"]["diag"][1])


def test_scalar_sigma_identity():
    wl = W.make_workload(1, n_blocks=2, block_size=2, n_energy=4)
    s = wl.sigma_s()
    assert np.allclose(s["g"]["value"] - s["l"]["value"], s["r"]["value"] - np.conj(s["r"]["value"]))


def test_offsets_config4():
    a = W.make_workload(4, n_blocks=3, block_size=4, n_energy=1)
    d = np.real(np.einsum("nii->ni", a.H_diag))
    assert np.abs(d).max() <= 3.0 + 6.0  # U[-1,1] + U[-2,2] + sqrt(2) Re CN tails / sqrt(b)
