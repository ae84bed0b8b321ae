"""Parity of the CUDA path with the oracle for the other populations of Eqs. 1-2 (
SURVEY.md 8(f) item 4): phonon-like (A = (w^2 + i eta) I - Phi, Bose-occupied contacts) and screened-Coulomb-like
(A = V^-1, B = P, no leads) inputs through the SAME C-ABI calls, by the input mappings stated in
paper_2602_03438_b200/workloads.py.  Bar: 1e-10 relative Frobenius error per block."""
import numpy as np
import pytest

from oracle import assemble, pipeline
from paper_2602_03438_b200 import workloads as W
from tests.helpers import rel_fro

pytestmark = pytest.mark.gpu
TOL = 1e-10

FAM = {"GR_diag": ("ret", "GR_diag"), "GR_upper": ("ret", "GR_upper"), "GR_lower": ("ret", "GR_lower"),
       "GL_diag": ("les", "GX_diag"), "GL_upper": ("les", "GX_upper"),
       "GG_diag": ("gtr", "GX_diag"), "GG_upper": ("gtr", "GX_upper")}


@pytest.fixture(scope="module")
def runner_mod(negf_lib):
    from paper_2602_03438_b200 import runner
    return runner


@pytest.mark.parametrize("n,b,nw", [(5, 24, 4), (4, 70, 3), (3, 130, 2)])
def test_phonon_like(runner_mod, n, b, nw):
    wl = W.make_phonon_workload(n, b, nw, periodic=False, seed=b)
    kT = 0.05
    outs, lefts, rights = [], [], []
    for k in range(nw):
        w2 = float(wl.energies[k])
        side = []
        for s in (0, 1):
            o = pipeline.obc_one_energy(w2, wl.eta, wl.H_diag, wl.H_upper, None, None, 0.0, kT, s, wl.tol, wl.max_iter)
            assert o["converged"]
            nb = 1.0 / np.expm1(np.sqrt(w2) / kT)                 # Bose occupation of the contact
            o["sigma_l"] = -1j * nb * o["gamma"]
            o["sigma_g"] = -1j * (nb + 1.0) * o["gamma"]
            side.append(o)
        lefts.append(side[0]); rights.append(side[1])
        outs.append(pipeline.solve_energy(wl, k, obc_in=(side[0], side[1]), want_greater=True))
    dp = runner_mod.DevicePath(wl, want_greater=True)
    # the decimation itself at z = w^2 + i eta, judged as in tests/test_gpu_path.py::test_obc_decimate (hazard H2: the
    # doublings are conditioning-limited): 1e-10 against the 80-bit oracle, else - labelled conditioning-limited,
    # never dropped - within 2x the largest error of the fp64 oracle ensemble (tests/helpers.fp64_oracle_ensemble)
    from tests.helpers import fp64_oracle_ensemble
    dp.obc()
    for s, (tag, ref) in enumerate((("L", lefts), ("R", rights))):
        sig = dp.host(f"sigma_r_{tag}")
        for k in range(nw):
            x = pipeline.obc_one_energy(float(wl.energies[k]), wl.eta, wl.H_diag, wl.H_upper, None, None, 0.0, kT, s,
                                        wl.tol, wl.max_iter, extended=True)["sigma_r"].astype(np.complex128)
            e = rel_fro(sig[k], x)
            if e > TOL:
                ens = fp64_oracle_ensemble(float(wl.energies[k]), wl.eta, wl.H_diag, wl.H_upper, None, None, s, wl.tol,
                                           wl.max_iter, seed=1000 * s + k)
                e_ref = max(rel_fro(s_, x) for s_ in ens)
                assert e <= 2 * e_ref, (tag, k, e, e_ref)
    assert dp.host("status_L").tolist() == [0] * nw and dp.host("status_R").tolist() == [0] * nw
    keys = ("sigma_r", "gamma", "sigma_l", "sigma_g")
    dp.set_boundary({k: np.stack([o[k] for o in lefts]) for k in keys}, {k: np.stack([o[k] for o in rights]) for k in keys})
    dp.retarded(); dp.lesser_greater(); dp.observables()
    assert dp.host("info_r").tolist() == [0] * nw
    for name, (grp, key) in FAM.items():
        assert rel_fro(dp.host(name), np.stack([o[grp][key] for o in outs])) < TOL, name
    T = np.array([o["obs"]["transmission"] for o in outs])
    assert np.allclose(dp.host("transmission"), T, rtol=1e-9, atol=1e-13)


@pytest.mark.parametrize("n,b,nw", [(4, 40, 3), (3, 130, 2), (1, 33, 2)])
def test_coulomb_like(runner_mod, n, b, nw):
    wl, sig = W.make_coulomb_workload(n, b, nw, seed=b)
    zero = {k: np.zeros((b, b), complex) for k in ("sigma_r", "gamma", "sigma_l", "sigma_g")}
    outs = []
    for k in range(nw):
        s1 = {t: {kk: (vv[k:k + 1] if kk != "kind" else vv) for kk, vv in sig[t].items()} for t in "rlg"}
        outs.append(pipeline.solve_energy(wl, k, sigma=s1, obc_in=(zero, zero), want_greater=True, corner=False))
    dp = runner_mod.DevicePath(wl, want_greater=True, sigma=sig)
    zb = {k: np.zeros((nw, b, b), complex) for k in zero}
    dp.set_boundary(zb, zb)
    dp.retarded(corner=False); dp.lesser_greater()
    assert dp.host("info_r").tolist() == [0] * nw
    for name, (grp, key) in FAM.items():
        ref = np.stack([o[grp][key] for o in outs])
        if ref.shape[1]:
            assert rel_fro(dp.host(name), ref) < TOL, name
    # and directly the Dyson equation with V itself: W^R = (I - V P^R)^-1 V
    h = lambda a: np.conj(np.swapaxes(a, -1, -2))
    V = np.linalg.inv(assemble.bt_to_dense(-wl.H_diag, -wl.H_upper, -h(wl.H_upper)))
    for k in range(nw):
        PR = assemble.bt_to_dense(sig["r"]["diag"][k], sig["r"]["upper"][k], sig["r"]["lower"][k])
        d, u, l = assemble.dense_to_bt(np.linalg.solve(np.eye(n * b) - V @ PR, V), n, b)
        assert rel_fro(dp.host("GR_diag")[k], d) < TOL
        if n > 1:
            assert rel_fro(dp.host("GR_upper")[k], u) < TOL and rel_fro(dp.host("GR_lower")[k], l) < TOL
