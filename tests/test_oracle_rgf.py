"""Pins for oracle/rgf.py, oracle/dense.py, oracle/assemble.py.
CPU only."""
import numpy as np
import pytest

from oracle import assemble, dense, pipeline, rgf
from paper_2602_03438_b200 import workloads as W
from tests.helpers import rel_fro

dag = assemble.dagger

CASES = [
    (0, {}),                                                  # configs[0] itself
    (0, dict(n_blocks=1, block_size=4)),                      # n = 1: no sweeps, both Sigma_B on one block
    (0, dict(n_blocks=2, block_size=1)),                      # n = 2, b = 1
    (0, dict(n_blocks=3, block_size=2)),
    (1, dict(n_blocks=4, block_size=5, n_energy=3)),          # scalar Sigma_S
    (2, dict(n_blocks=5, block_size=6, n_energy=2)),          # S != I
    (3, dict(n_blocks=4, block_size=8, n_energy=3)),          # BT Sigma^{R,<,>}
    (3, dict(n_blocks=2, block_size=3, n_energy=2)),
    (4, dict(n_blocks=3, block_size=7, n_energy=2)),          # offsets
]


def _solve(cfg, kw, k):
    wl = W.make_workload(cfg, **kw)
    if wl.n_blocks == 1:
        # decimation with periodic copies needs n >= 2: feed explicit Sigma_B
        rng = np.random.default_rng(5)
        b = wl.block_size
        def lead(f):
            m = W.complex_normal(rng, (b, b), 0.1)
            sig = -1j * (m @ dag(m)) + 0.05 * (m + dag(m))
            gam = 1j * (sig - dag(sig))
            return {"sigma_r": sig, "gamma": gam, "sigma_l": 1j * f * gam, "sigma_g": -1j * (1 - f) * gam, "f": f}
        return wl, pipeline.solve_energy(wl, k, obc_in=(lead(0.7), lead(0.2)), want_greater=True)
    return wl, pipeline.solve_energy(wl, k, want_greater=True)


@pytest.mark.parametrize("cfg,kw", CASES)
def test_rgf_equals_dense_definition(cfg, kw):
    """P1: every selected block of tier 1 equals the dense definition."""
    wl = W.make_workload(cfg, **kw)
    for k in range(wl.n_energy):
        wl, out = _solve(cfg, kw, k)
        n, b = wl.n_blocks, wl.block_size
        d = dense.dense_green(*out["A"], B_list=[out["BL"], out["BG"]])
        r = out["ret"]
        tol = 2e-11
        assert rel_fro(r["GR_diag"], d["GR"][0]) < tol
        if n > 1:
            assert rel_fro(r["GR_upper"], d["GR"][1]) < tol
            assert rel_fro(r["GR_lower"], d["GR"][2]) < tol
        assert rel_fro(r["GR_corner"][0], d["GR_full"][:b, (n - 1) * b:]) < tol
        for name, j in (("les", 0), ("gtr", 1)):
            assert rel_fro(out[name]["GX_diag"], d["GX"][j][0]) < tol
            if n > 1:
                assert rel_fro(out[name]["GX_upper"], d["GX"][j][1]) < tol
                assert rel_fro(out[name]["GX_lower"], d["GX"][j][2]) < tol


def test_config0_extended_precision():
    """P1: configs[0] against 80-bit Gauss-Jordan dense inversion (fp64 LAPACK not trusted alone)."""
    wl, out = _solve(0, {}, 0)
    d64 = dense.dense_green(*out["A"], B_list=[out["BL"]])
    d80 = dense.dense_green(*out["A"], B_list=[out["BL"]], extended=True)
    # the extended inverse really is an inverse, to extended accuracy
    A80 = assemble.bt_to_dense(*[x.astype(np.clongdouble) for x in out["A"]])
    res = np.abs(A80 @ d80["GR_full"] - np.eye(A80.shape[0])).max()
    assert res < 1e-15
    for j in range(3):
        assert rel_fro(d64["GR"][j], d80["GR"][j].astype(np.complex128)) < 1e-11
        assert rel_fro(out["ret"][("GR_diag", "GR_upper", "GR_lower")[j]], d80["GR"][j].astype(np.complex128)) < 1e-11
    assert rel_fro(out["les"]["GX_diag"], d80["GX"][0][0].astype(np.complex128)) < 1e-10
    assert rel_fro(out["les"]["GX_upper"], d80["GX"][0][1].astype(np.complex128)) < 1e-10


def test_hand_solved_2x2():
    """P10 brute force: n = 2, b = 1, inverse and triple product written out by hand."""
    a, u, l, d = 0.3 + 0.2j, -0.7 + 0.1j, 0.4 - 0.5j, -0.2 + 0.6j
    p, q, r = 0.9j, 0.3 - 0.2j, 0.4j            # B = [[p, q], [-conj(q), r]] anti-Hermitian
    det = a * d - u * l
    G = np.array([[d, -u], [-l, a]]) / det
    B = np.array([[p, q], [-np.conj(q), r]])
    GX = G @ B @ G.conj().T
    A_diag = np.array([[[a]], [[d]]]); A_up = np.array([[[u]]]); A_lo = np.array([[[l]]])
    ret = rgf.rgf_retarded(A_diag, A_up, A_lo, corner=True)
    les = rgf.rgf_lesser_greater(A_up, A_lo, np.array([[[p]], [[r]]]), np.array([[[q]]]), ret)
    assert np.allclose(ret["GR_diag"][:, 0, 0], [G[0, 0], G[1, 1]], rtol=1e-14)
    assert np.allclose(ret["GR_upper"][0, 0, 0], G[0, 1], rtol=1e-14)
    assert np.allclose(ret["GR_lower"][0, 0, 0], G[1, 0], rtol=1e-14)
    assert np.allclose(ret["GR_corner"][0, 0, 0], G[0, 1], rtol=1e-14)
    assert np.allclose(les["GX_diag"][:, 0, 0], [GX[0, 0], GX[1, 1]], rtol=1e-13)
    assert np.allclose(les["GX_upper"][0, 0, 0], GX[0, 1], rtol=1e-13)
    assert np.allclose(les["GX_lower"][0, 0, 0], GX[1, 0], rtol=1e-13)


def test_hand_solved_1x1():
    """P10: n = 1, b = 1: G = 1/a, G^< = B/|a|^2."""
    a, p = 0.3 - 0.4j, 0.25j
    ret = rgf.rgf_retarded(np.array([[[a]]]), np.zeros((0, 1, 1), complex), np.zeros((0, 1, 1), complex))
    les = rgf.rgf_lesser_greater(np.zeros((0, 1, 1), complex), np.zeros((0, 1, 1), complex),
                                 np.array([[[p]]]), np.zeros((0, 1, 1), complex), ret)
    assert np.isclose(ret["GR_diag"][0, 0, 0], 1 / a)
    assert np.isclose(les["GX_diag"][0, 0, 0], p / abs(a) ** 2)


@pytest.mark.parametrize("cfg,kw", [CASES[0], CASES[6], CASES[5]])
def test_selected_block_residuals(cfg, kw):
    """P2/P3: Eq. 1 and Eq. 2 residuals from the selected blocks only."""
    wl, out = _solve(cfg, kw, 0)
    Ad, Au, Al = out["A"]
    r, les = out["ret"], out["les"]
    Bd, Bu = out["BL"]
    n, b = wl.n_blocks, wl.block_size
    for i in range(n):
        # (A G)_ii = I
        acc = Ad[i] @ r["GR_diag"][i]
        if i > 0:
            acc += Al[i - 1] @ r["GR_upper"][i - 1]
        if i + 1 < n:
            acc += Au[i] @ r["GR_lower"][i]
        assert np.abs(acc - np.eye(b)).max() < 1e-9
        # (A G^<)_ii = sum_j B_ij (G^R_ij)^H over the BT pattern
        lhs = Ad[i] @ les["GX_diag"][i]
        rhs = Bd[i] @ dag(r["GR_diag"][i])
        if i > 0:
            lhs += Al[i - 1] @ les["GX_upper"][i - 1]
            rhs += (-dag(Bu[i - 1])) @ dag(r["GR_lower"][i - 1])     # B_{i,i-1} (G_{i,i-1})^H
        if i + 1 < n:
            lhs += Au[i] @ les["GX_lower"][i]
            rhs += Bu[i] @ dag(r["GR_upper"][i])                     # B_{i,i+1} (G_{i,i+1})^H
        assert np.abs(lhs - rhs).max() < 1e-9 * max(1.0, np.abs(rhs).max())


@pytest.mark.parametrize("cfg,kw", [CASES[6], CASES[4]])
def test_cross_checks_of_8c1(cfg, kw):
    """independent lower block and six-term diagonal form agree with S6."""
    wl, out = _solve(cfg, kw, 1)
    _, Au, Al = out["A"]
    for name, B in (("les", out["BL"]), ("gtr", out["BG"])):
        for i in range(wl.n_blocks - 1):
            low = rgf.lower_block_independent(Au, Al, B[1], out["ret"], out[name], i)
            assert rel_fro(low, out[name]["GX_lower"][i]) < 1e-10
            six = rgf.diag_block_six_terms(Au, Al, B[1], out["ret"], out[name], i)
            assert rel_fro(six, out[name]["GX_diag"][i]) < 1e-10


@pytest.mark.parametrize("cfg,kw", [CASES[0], CASES[6], CASES[4]])
def test_symmetries_and_corrected_spectral_identity(cfg, kw):
    """P4 + hazard H1: (G^x)^H = -G^x; G^> - G^< = G^R - G^A + 2 i eta G^R S G^A (dense, tiny)."""
    wl, out = _solve(cfg, kw, 0)
    for name in ("les", "gtr"):
        for blk in out[name]["GX_diag"]:
            assert np.abs(blk + dag(blk)).max() < 1e-10 * max(np.abs(blk).max(), 1e-300)
    d = dense.dense_green(*out["A"], B_list=[out["BL"], out["BG"]])
    GR = d["GR_full"]
    n, b = wl.n_blocks, wl.block_size
    if wl.S_diag is None:
        S = np.eye(n * b)
    else:
        S = assemble.bt_to_dense(wl.S_diag, wl.S_upper, dag(wl.S_upper))
    lhs = d["GX_full"][1] - d["GX_full"][0]
    rhs = GR - dag(GR) + 2j * wl.eta * GR @ S @ dag(GR)
    assert np.linalg.norm(lhs - rhs) / np.linalg.norm(rhs) < 1e-9
    # and the same identity on the RGF selected blocks
    rd = assemble.dense_to_bt(rhs, n, b)
    assert rel_fro(out["gtr"]["GX_diag"] - out["les"]["GX_diag"], rd[0]) < 1e-8


def test_gauss_jordan_matches_lapack():
    rng = np.random.default_rng(3)
    M = rng.standard_normal((9, 9)) + 1j * rng.standard_normal((9, 9))
    assert np.allclose(dense.gauss_jordan_inverse(M), np.linalg.inv(M), rtol=1e-11, atol=1e-12)


@pytest.mark.parametrize("k", [0, 37])
def test_config1_full_size_rgf_equals_dense(k):
    """P1 at the size bench.py times: configs[1] (n = 32, b = 64, N = 2048, scalar scattering), tier 1 against
    the dense fp64 definition for two energies of the grid."""
    wl = W.make_workload(1)
    out = pipeline.solve_energy(wl, k, want_greater=False)
    d = dense.dense_green(*out["A"], B_list=[out["BL"]])
    r = out["ret"]
    tol = 5e-10            # cond(A) ~ 1e3-1e4 at this size; both sides are fp64
    assert rel_fro(r["GR_diag"], d["GR"][0]) < tol
    assert rel_fro(r["GR_upper"], d["GR"][1]) < tol
    assert rel_fro(r["GR_lower"], d["GR"][2]) < tol
    assert rel_fro(r["GR_corner"][0], d["GR_full"][:64, 31 * 64:]) < tol
    assert rel_fro(out["les"]["GX_diag"], d["GX"][0][0]) < tol
    assert rel_fro(out["les"]["GX_upper"], d["GX"][0][1]) < tol
