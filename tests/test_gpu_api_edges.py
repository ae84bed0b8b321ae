"""C-ABI edge behaviour on the GPU: optional outputs left out (NULL), a non-default stream, error codes,
per-energy numerical failure codes."""
import numpy as np
import pytest
import torch

from oracle import pipeline
from paper_2602_03438_b200 import workloads as W
from tests.helpers import rel_fro

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def runner_mod(negf_lib):
    from paper_2602_03438_b200 import runner
    return runner


@pytest.mark.parametrize("cfg,kw", [(1, dict(n_blocks=7, block_size=24, n_energy=3)),      # two-sided path
                                    (4, dict(n_blocks=4, block_size=130, n_energy=2))])    # one-sided path
def test_optional_outputs_null(runner_mod, negf_lib, cfg, kw):
    """GR_upper / GR_lower / GR_corner / G^x_upper may be NULL: the diagonal blocks must not change."""
    wl = W.make_workload(cfg, **kw)
    dp = runner_mod.DevicePath(wl, want_greater=True)
    dp.run()
    full = {k: dp.host(k).copy() for k in ("GR_diag", "GL_diag", "GG_diag")}
    o = dp.out
    for k in ("GR_diag", "GL_diag", "GG_diag"):
        o[k].zero_()
    sr = dp._sigma("r", o["sigma_r_L"], o["sigma_r_R"])
    info = torch.zeros(wl.n_energy, dtype=torch.int32, device="cuda")
    dp.ctx.rgf_retarded(dp.problem, sr, o["GR_diag"], None, None, None, negf_lib.KEEP_SWEEP, info)
    sl = dp._sigma("l", o["sigma_l_L"], o["sigma_l_R"])
    sg = dp._sigma("g", o["sigma_g_L"], o["sigma_g_R"])
    dp.ctx.rgf_lesser_greater(dp.problem, sr, sl, sg, o["GR_diag"], o["GL_diag"], None, o["GG_diag"], None, info)
    for k, v in full.items():
        assert rel_fro(dp.host(k), v) < 1e-13, k
    # only G^< requested
    o["GL_diag"].zero_()
    dp.ctx.rgf_lesser_greater(dp.problem, sr, sl, None, o["GR_diag"], o["GL_diag"], None, None, None, info)
    assert rel_fro(dp.host("GL_diag"), full["GL_diag"]) < 1e-13


def test_non_default_stream(runner_mod):
    """All work goes to the stream given by negf_set_stream; results match the oracle."""
    wl = W.make_workload(1, n_blocks=5, block_size=32, n_energy=4)
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        dp = runner_mod.DevicePath(wl, want_greater=False)
        for _ in range(3):          # plain, captured, replayed
            dp.run()
    st.synchronize()
    for k in (0, 3):
        side = lambda t: {"sigma_r": dp.host(f"sigma_r_{t}")[k], "gamma": dp.host(f"gamma_{t}")[k],
                          "sigma_l": dp.host(f"sigma_l_{t}")[k], "sigma_g": dp.host(f"sigma_g_{t}")[k]}
        o = pipeline.solve_energy(wl, k, obc_in=(side("L"), side("R")), want_greater=False)
        assert rel_fro(dp.host("GR_diag")[k], o["ret"]["GR_diag"]) < 1e-10
        assert rel_fro(dp.host("GL_upper")[k], o["les"]["GX_upper"]) < 1e-10


def test_error_codes(runner_mod, negf_lib):
    wl = W.make_workload(0)
    dp = runner_mod.DevicePath(wl, want_greater=True)
    o = dp.out
    sr = dp._sigma("r", o["sigma_r_L"], o["sigma_r_R"])
    sl = dp._sigma("l", o["sigma_l_L"], o["sigma_l_R"])
    # lesser/greater without retained sweep state
    dp.ctx.set_workspace(dp.workspace)           # drops any state
    rc = negf_lib.lib.negf_rgf_lesser_greater(dp.ctx._h, dp.problem, sr, sl, None, o["GR_diag"].data_ptr(),
                                              o["GL_diag"].data_ptr(), None, None, None, o["info_x"].data_ptr())
    assert rc == negf_lib.ENOSTATE
    # workspace too small
    small = torch.empty(1024, dtype=torch.uint8, device="cuda")
    dp.ctx.set_workspace(small)
    rc = negf_lib.lib.negf_rgf_retarded(dp.ctx._h, dp.problem, sr, o["GR_diag"].data_ptr(), None, None, None, 0,
                                        o["info_r"].data_ptr())
    assert rc == negf_lib.ENOWORKSPACE
    # misaligned workspace, bad side, missing required output
    assert negf_lib.lib.negf_set_workspace(dp.ctx._h, dp.workspace.data_ptr() + 8, 1 << 20) == negf_lib.EINVAL
    dp.ctx.set_workspace(dp.workspace)
    rc = negf_lib.lib.negf_obc_decimate(dp.ctx._h, dp.problem, None, 2, 0.0, 0.025, 1e-12, 64,
                                        o["sigma_r_L"].data_ptr(), None, None, None, None, None,
                                        o["iters_L"].data_ptr(), o["status_L"].data_ptr())
    assert rc == negf_lib.EINVAL
    rc = negf_lib.lib.negf_rgf_retarded(dp.ctx._h, dp.problem, sr, None, None, None, None, 0, o["info_r"].data_ptr())
    assert rc == negf_lib.EINVAL
    assert negf_lib.lib.negf_set_option(dp.ctx._h, 12345, 1) == negf_lib.EINVAL


@pytest.mark.parametrize("b", [12, 130])
def test_singular_block_is_reported_per_energy(runner_mod, negf_lib, b):
    """A zero diagonal block at the start of the sweep (energy 1 only) sets info[1] = 1 (block 0, LAPACK style)
    and leaves the other energies untouched."""
    wl = W.make_workload(0, n_blocks=1, block_size=b, n_energy=1)
    wl.energies = np.array([0.3, 0.5, 0.7]); wl.weights = np.ones(3)
    wl.H_diag[0] = np.diag(np.full(b, 0.5)).astype(complex)
    wl.eta = 0.0                                     # z - H = 0 exactly at E = 0.5
    dp = runner_mod.DevicePath(wl, want_greater=False)
    zero = torch.zeros(3, b, b, dtype=torch.complex128, device="cuda")
    sr = negf_lib.make_sigma(negf_lib.SIGMA_NONE, left=zero, right=zero)
    dp.ctx.rgf_retarded(dp.problem, sr, dp.out["GR_diag"], None, None, None, 0, dp.out["info_r"])
    info = dp.host("info_r").tolist()
    assert info[0] == 0 and info[2] == 0 and info[1] == 1
    g = dp.host("GR_diag")
    assert np.allclose(g[0, 0], np.eye(b) / (0.3 - 0.5)) and np.allclose(g[2, 0], np.eye(b) / (0.7 - 0.5))
