"""Momentum (k-point) batching ("the momentum dependence is omitted for simplicity"; SURVEY.md 8(f)
item 2): one call takes n_k devices H(k), S(k) and a list of (k, E) batch entries and runs them as ONE lock-step
batch.  The oracle is a plain loop over k of the single-device path; comparison per block at the 1e-10 bar with the
oracle's boundary blocks fed to the GPU (hazard H2), as in tests/test_gpu_path.py."""
import numpy as np
import pytest
import torch

from oracle import pipeline
from paper_2602_03438_b200 import workloads as W
from tests.helpers import rel_fro

pytestmark = pytest.mark.gpu
TOL = 1e-10

CASES = [(1, 3, dict(n_blocks=6, block_size=24, n_energy=4)),       # two-sided path, scalar Sigma_S
         (2, 3, dict(n_blocks=4, block_size=40, n_energy=3)),       # S(k) != I
         (3, 2, dict(n_blocks=4, block_size=72, n_energy=2)),       # dense BT Sigma_S, kernel 65..96
         (4, 2, dict(n_blocks=3, block_size=130, n_energy=2)),      # one-sided path, blocked inverse
         (1, 4, dict(n_blocks=5, block_size=16, n_energy=12))]      # 48 entries: 4 energy groups crossing k boundaries


def _oracle(wls, want_greater=True):
    outs = []
    for wl in wls:
        sig = wl.sigma_s()
        for e in range(wl.n_energy):
            s1 = {t: (None if sig[t] is None else {kk: (vv[e:e + 1] if kk != "kind" else vv) for kk, vv in sig[t].items()})
                  for t in "rlg"}
            outs.append(pipeline.solve_energy(wl, e, sigma=s1, want_greater=want_greater))
    return outs


@pytest.mark.parametrize("cfg,nk,kw", CASES)
def test_kpoint_batch_against_oracle_loop(negf_lib, cfg, nk, kw):
    from paper_2602_03438_b200 import runner
    wls, ks, wk = W.make_kpoint_workloads(cfg, nk, **kw)
    outs = _oracle(wls)
    dp = runner.DevicePath(wls[0], want_greater=True, kpoints=wls, k_weights=wk)
    assert dp.ne == nk * wls[0].n_energy
    # (1) the whole path in one call: decimation of every (k, E) entry, iteration counts as the oracle's
    dp.run()
    torch.cuda.synchronize()
    for tag, side in (("L", "left"), ("R", "right")):
        assert dp.host(f"status_{tag}").tolist() == [0] * dp.ne
        its = np.array([o[side]["iters"] for o in outs])
        assert np.max(np.abs(dp.host(f"iters_{tag}") - its)) <= 1                    # reading R3
        ref = np.stack([o[side]["sigma_r"] for o in outs])
        assert rel_fro(dp.host(f"sigma_r_{tag}"), ref) < 1e-6                        # conditioning-limited (H2): loose here
    e2e = rel_fro(dp.host("GR_diag"), np.stack([o["ret"]["GR_diag"] for o in outs]))
    assert e2e < 1e-5, e2e
    # (2) identical boundary blocks -> the 1e-10 bar on every family
    stack = lambda side, key: np.stack([o[side][key] for o in outs])
    keys = ("sigma_r", "gamma", "sigma_l", "sigma_g")
    dp.set_boundary({k: stack("left", k) for k in keys}, {k: stack("right", k) for k in keys})
    dp.retarded(); dp.lesser_greater(); dp.observables()
    torch.cuda.synchronize()
    assert dp.host("info_r").tolist() == [0] * dp.ne
    fam = {"GR_diag": ("ret", "GR_diag"), "GR_upper": ("ret", "GR_upper"), "GR_lower": ("ret", "GR_lower"),
           "GL_diag": ("les", "GX_diag"), "GL_upper": ("les", "GX_upper"),
           "GG_diag": ("gtr", "GX_diag"), "GG_upper": ("gtr", "GX_upper")}
    for name, (grp, key) in fam.items():
        err = rel_fro(dp.host(name), np.stack([o[grp][key] for o in outs]))
        assert err < TOL, (name, err)
    assert rel_fro(dp.host("GR_corner"), np.stack([o["ret"]["GR_corner"][0] for o in outs])) < TOL
    T = np.array([o["obs"]["transmission"] for o in outs])
    assert np.allclose(dp.host("transmission"), T, rtol=1e-9, atol=1e-13)
    ld = np.stack([o["obs"]["ldos"] for o in outs])
    assert np.allclose(dp.host("ldos"), ld, rtol=1e-9, atol=1e-12 * np.abs(ld).max())
    # density: sum over k and E with weights w_k w_E, each entry with the overlap S(k) of ITS device
    ne1 = wls[0].n_energy
    dens = sum(wk[j] * pipeline.density(wls[j], [outs[j * ne1 + e]["obs"]["density_integrand"] for e in range(ne1)])
               for j in range(nk))
    assert np.allclose(dp.host("density"), dens, rtol=1e-9, atol=1e-12 * np.abs(dens).max())
    J = np.stack([o["obs"]["bond_current"] for o in outs])
    n = wls[0].n_blocks
    for q, o in enumerate(outs):
        wl = wls[q // ne1]
        for i in range(n - 1):
            hop = wl.H_upper[i] if wl.S_upper is None else wl.H_upper[i] - wl.energies[q % ne1] * wl.S_upper[i]
            scale = 2 * np.linalg.norm(hop) * np.linalg.norm(o["les"]["GX_upper"][i])
            assert abs(dp.host("bond_current")[q, i] - J[q, i]) <= TOL * scale + 1e-300


def test_kpoint_batch_equals_separate_calls(negf_lib):
    """The k-batched call against one call per k-point on the same library: same arithmetic per entry (the
    launch shapes differ with the batch size, so agreement is to rounding, not to the bit)."""
    from paper_2602_03438_b200 import runner
    wls, ks, wk = W.make_kpoint_workloads(1, 3, n_blocks=5, block_size=32, n_energy=5)
    dp = runner.DevicePath(wls[0], want_greater=True, kpoints=wls, k_weights=wk)
    dp.run()
    torch.cuda.synchronize()
    ne1 = wls[0].n_energy
    dens = 0.0
    for j, wl in enumerate(wls):
        one = runner.DevicePath(wl, want_greater=True)
        one.run()
        torch.cuda.synchronize()
        for name in ("sigma_r_L", "sigma_r_R", "GR_diag", "GR_upper", "GL_diag", "GL_upper", "GG_diag"):
            assert rel_fro(dp.host(name)[j * ne1:(j + 1) * ne1], one.host(name)) < 1e-9, (j, name)   # decimation: H2
        assert np.allclose(dp.host("transmission")[j * ne1:(j + 1) * ne1], one.host("transmission"), rtol=1e-7)
        dens = dens + wk[j] * one.host("density")
    assert np.allclose(dp.host("density"), dens, rtol=1e-7, atol=1e-10 * np.abs(dens).max())


def test_kpoint_batch_through_the_host_pipeline(negf_lib):
    """negf_pipeline_host with n_k > 1 (HOST k_index) against negf_pipeline_device on the same batch."""
    from paper_2602_03438_b200 import runner
    wls, ks, wk = W.make_kpoint_workloads(2, 2, n_blocks=4, block_size=24, n_energy=3)
    hp = runner.HostPath(wls[0], want_greater=True, kpoints=wls, k_weights=wk)
    hp.run()
    assert hp.out["info"].tolist() == [0] * hp.ne
    dp = runner.DevicePath(wls[0], want_greater=True, kpoints=wls, k_weights=wk)
    dp.run()
    torch.cuda.synchronize()
    for nm in ("GR_diag", "GR_upper", "GR_lower", "GL_diag", "GL_upper", "GG_diag", "GG_upper"):
        assert rel_fro(hp.out[nm].numpy(), dp.host(nm)) < 1e-12, nm
    d = dp.host("density")
    assert np.allclose(hp.out["density"].numpy(), d, rtol=1e-10, atol=1e-12 * np.abs(d).max())


def test_kpoint_arguments_are_checked(negf_lib):
    from paper_2602_03438_b200 import runner
    wls, ks, wk = W.make_kpoint_workloads(1, 2, n_blocks=3, block_size=8, n_energy=2)
    dp = runner.DevicePath(wls[0], want_greater=False, kpoints=wls, k_weights=wk)
    p = dp.problem
    bad = negf_lib.Problem(p.n_blocks, p.block_size, p.n_energy, p.H_diag, p.H_upper, p.S_diag, p.S_upper, p.energy,
                           p.eta, 2, None)                       # n_k > 1 without k_index
    o = dp.out
    rc = negf_lib.lib.negf_rgf_retarded(dp.ctx._h, bad, None, o["GR_diag"].data_ptr(), None, None, None, 0,
                                        o["info_r"].data_ptr())
    assert rc == negf_lib.EINVAL
