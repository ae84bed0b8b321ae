"""Resident small-block regime (b <= 32, NEGF_OPT_FUSED_SMALL, csrc/fused_small.cu): the whole chain of one energy in
one CTA.  Every parity test of tests/test_gpu_path.py with b <= 32 already runs through it (it is the default);
here it is compared with the batched lock-step path of the same library (option 0) on the same inputs, for every
Sigma kind, ragged block sizes, n = 1 and n = 2, and k-point batches; and against the oracle at configs[0]."""
import numpy as np
import pytest
import torch

from oracle import pipeline
from paper_2602_03438_b200 import workloads as W
from tests.helpers import rel_fro

pytestmark = pytest.mark.gpu

CASES = [(0, {}), (0, dict(n_blocks=2, block_size=5)), (0, dict(n_blocks=3, block_size=1, n_energy=3)),
         (1, dict(n_blocks=6, block_size=24, n_energy=5)), (1, dict(n_blocks=9, block_size=32, n_energy=3)),
         (2, dict(n_blocks=4, block_size=17, n_energy=3)), (3, dict(n_blocks=4, block_size=31, n_energy=2)),
         (4, dict(n_blocks=3, block_size=8, n_energy=40))]


@pytest.mark.parametrize("cfg,kw", CASES)
def test_resident_path_equals_batched_path(negf_lib, cfg, kw):
    from paper_2602_03438_b200 import runner
    wl = W.make_workload(cfg, **kw)
    fused = runner.DevicePath(wl, want_greater=True)
    fused.run_four_calls()
    plain = runner.DevicePath(wl, want_greater=True)
    plain.ctx.set_option(negf_lib.OPT_FUSED_SMALL, 0)
    plain.run_four_calls()
    torch.cuda.synchronize()
    assert fused.ctx.launch_count() < 20 and plain.ctx.launch_count() > 3 * fused.ctx.launch_count()
    for tag in "LR":
        assert fused.host(f"status_{tag}").tolist() == [0] * wl.n_energy
        assert np.max(np.abs(fused.host(f"iters_{tag}") - plain.host(f"iters_{tag}"))) <= 1
        assert np.array_equal(fused.host(f"fermi_{tag}"), plain.host(f"fermi_{tag}"))
    # same boundary blocks for both -> the sweeps agree to rounding
    for k in ("sigma_r", "gamma", "sigma_l", "sigma_g"):
        for tag in "LR":
            plain.out[f"{k}_{tag}"].copy_(fused.out[f"{k}_{tag}"])
    for dp in (fused, plain):
        dp.retarded(); dp.lesser_greater(); dp.observables()
    torch.cuda.synchronize()
    # The two regimes eliminate in different orders (one-sided here, two-sided there), so where a Schur complement
    # of a sub-chain is nearly singular they differ by more than rounding of a well-conditioned problem (hazard H3):
    # loose bar between the paths, the 1e-10 / ensemble rule of tests/test_gpu_fullsize.py against the oracle.
    for nm in ("GR_diag", "GR_upper", "GR_lower", "GR_corner", "GL_diag", "GL_upper", "GG_diag", "GG_upper"):
        if fused.out[nm].numel() == 0:
            continue
        assert rel_fro(fused.host(nm), plain.host(nm)) < 1e-7, nm
    assert np.allclose(fused.host("transmission"), plain.host("transmission"), rtol=1e-7, atol=1e-13)
    from tests.helpers import rgf_oracle_ensemble
    sig = wl.sigma_s()
    for k in sorted({0, wl.n_energy // 2, wl.n_energy - 1}):
        side = lambda t: {"sigma_r": fused.host(f"sigma_r_{t}")[k], "gamma": fused.host(f"gamma_{t}")[k],
                          "sigma_l": fused.host(f"sigma_l_{t}")[k], "sigma_g": fused.host(f"sigma_g_{t}")[k]}
        s1 = {t: (None if sig[t] is None else {kk: (vv[k:k + 1] if kk != "kind" else vv) for kk, vv in sig[t].items()})
              for t in "rlg"}
        o = pipeline.solve_energy(wl, k, sigma=s1, obc_in=(side("L"), side("R")), want_greater=True)
        ens = None
        fams = [("GR_diag", o["ret"]["GR_diag"], lambda m: m["GR_diag"]), ("GR_upper", o["ret"]["GR_upper"], lambda m: m["GR_upper"]),
                ("GL_diag", o["les"]["GX_diag"], lambda m: m["GX"][0][0]), ("GL_upper", o["les"]["GX_upper"], lambda m: m["GX"][0][1]),
                ("GG_diag", o["gtr"]["GX_diag"], lambda m: m["GX"][1][0]), ("GG_upper", o["gtr"]["GX_upper"], lambda m: m["GX"][1][1])]
        for nm, ref, pick in fams:
            if ref.shape[0] == 0:
                continue
            e = rel_fro(fused.host(nm)[k], ref)
            if e > 1e-10:
                if ens is None:
                    ens = rgf_oracle_ensemble(o["A"], [o["BL"], o["BG"]], seed=k)
                spread = max(rel_fro(pick(m), ref) for m in ens)
                assert e <= 3 * spread, (k, nm, e, spread)         # H3 rule of tests/test_gpu_fullsize.py


def test_resident_path_kpoints_and_option_switch(negf_lib):
    """k-point batches run through the resident kernels too; switching the option drops the retained state."""
    from paper_2602_03438_b200 import runner
    wls, ks, wk = W.make_kpoint_workloads(2, 3, n_blocks=4, block_size=12, n_energy=3)
    a = runner.DevicePath(wls[0], want_greater=True, kpoints=wls, k_weights=wk)
    a.run()
    b = runner.DevicePath(wls[0], want_greater=True, kpoints=wls, k_weights=wk)
    b.ctx.set_option(negf_lib.OPT_FUSED_SMALL, 0)
    b.run()
    torch.cuda.synchronize()
    for nm in ("sigma_r_L", "sigma_r_R", "GR_diag", "GL_diag", "GG_upper"):
        assert rel_fro(a.host(nm), b.host(nm)) < 1e-8, nm          # decimation is conditioning-limited (H2)
    # retained state of one regime is not valid for the other
    a.retarded()
    a.ctx.set_option(negf_lib.OPT_FUSED_SMALL, 0)
    with pytest.raises(negf_lib.NegfError):
        a.lesser_greater()


def test_config0_latency(negf_lib):
    """configs[0] (one energy, n = 8, b = 16) through negf_pipeline_device: a handful of launches, and the RGF at the
    1e-10 bar against the oracle fed with the same boundary blocks."""
    from paper_2602_03438_b200 import runner
    wl = W.make_workload(0)
    dp = runner.DevicePath(wl, want_greater=True)
    dp.run(); torch.cuda.synchronize()
    l0 = dp.ctx.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(20):
        dp.run()
    e1.record(); torch.cuda.synchronize()
    per = (dp.ctx.launch_count() - l0) / 20
    us = e0.elapsed_time(e1) * 1e3 / 20
    print(f"configs[0] whole path: {us:.1f} us per pass, {per:.0f} kernel launches")
    assert per < 20
    k = 0
    side = lambda t: {"sigma_r": dp.host(f"sigma_r_{t}")[k], "gamma": dp.host(f"gamma_{t}")[k],
                      "sigma_l": dp.host(f"sigma_l_{t}")[k], "sigma_g": dp.host(f"sigma_g_{t}")[k]}
    o = pipeline.solve_energy(wl, 0, obc_in=(side("L"), side("R")), want_greater=True)
    for nm, grp, key in (("GR_diag", "ret", "GR_diag"), ("GR_upper", "ret", "GR_upper"), ("GL_diag", "les", "GX_diag"),
                         ("GL_upper", "les", "GX_upper"), ("GG_diag", "gtr", "GX_diag")):
        assert rel_fro(dp.host(nm)[0], o[grp][key]) < 1e-10, nm


@pytest.mark.parametrize("cfg,kw", [(0, {}), (1, dict(n_blocks=9, block_size=32, n_energy=150)),
                                    (2, dict(n_blocks=5, block_size=17, n_energy=300)), (3, dict(n_blocks=4, block_size=31, n_energy=20))])
def test_resident_path_is_bit_identical_run_to_run(negf_lib, cfg, kw):
    """The resident kernels hand data between warps through named barriers, shuffles, an mbarrier and double-buffered
    shared memory; every reduction has a fixed order.  A race would show as a run-to-run difference: twelve passes of
    the whole path must reproduce the first one bit for bit (one wave and more than one wave of CTAs, every Sigma kind)."""
    from paper_2602_03438_b200 import runner
    wl = W.make_workload(cfg, **kw)
    dp = runner.DevicePath(wl, want_greater=True)
    dp.run(); torch.cuda.synchronize()
    ref = {k: v.clone() for k, v in dp.out.items()}
    for rep in range(12):
        dp.run()
        torch.cuda.synchronize()
        for k, v in dp.out.items():
            a = torch.view_as_real(v) if v.is_complex() else v
            r = torch.view_as_real(ref[k]) if ref[k].is_complex() else ref[k]
            assert torch.equal(torch.nan_to_num(a.double()), torch.nan_to_num(r.double())), (k, rep)


@pytest.mark.parametrize("cfg,kw", [(0, {}), (1, dict(n_blocks=5, block_size=24, n_energy=4)),
                                    (2, dict(n_blocks=4, block_size=17, n_energy=3)), (2, dict(n_blocks=2, block_size=9, n_energy=40)),
                                    (3, dict(n_blocks=3, block_size=32, n_energy=2))])
def test_resident_observables_equal_batched_kernels(negf_lib, cfg, kw):
    """S7 of the resident regime is ONE launch (observables.cu:obs_small_kernel, blocks take roles); fed with the SAME G
    blocks and boundary blocks it must reproduce the seven separate kernels of the batched path to summation order
    (S != I exercises the three-term density and LDOS, configs[2])."""
    from paper_2602_03438_b200 import runner
    wl = W.make_workload(cfg, **kw)
    fused = runner.DevicePath(wl, want_greater=True)
    fused.run_four_calls()
    plain = runner.DevicePath(wl, want_greater=True)
    plain.ctx.set_option(negf_lib.OPT_FUSED_SMALL, 0)
    plain.run_four_calls()                                   # sizes the workspace the batched T(E) needs
    torch.cuda.synchronize()
    for k, v in fused.out.items():
        if k not in ("density", "ldos", "transmission", "bond_current", "contact_current"):
            plain.out[k].copy_(v)
    n0 = fused.ctx.launch_count()
    fused.observables()
    assert fused.ctx.launch_count() - n0 == 1
    plain.observables()
    torch.cuda.synchronize()
    names = ["density", "ldos", "transmission", "contact_current"] + (["bond_current"] if wl.n_blocks > 1 else [])
    for nm in names:
        a, b = fused.host(nm), plain.host(nm)
        scale = np.max(np.abs(b)) + 1e-300
        assert np.max(np.abs(a - b)) <= 1e-12 * scale + 1e-13 * np.max(np.abs(fused.host("GL_diag"))), (nm, np.max(np.abs(a - b)), scale)
