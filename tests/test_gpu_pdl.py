"""Programmatic dependent launch of the chain kernels (NEGF_OPT_PDL, csrc/common.cuh): the K2 small-tile kernel, the
one-CTA inverse and the decimation step are launched with the programmatic-stream-serialization attribute and wait
for the previous kernel with griddepcontrol.wait.  The attribute changes WHEN a kernel's CTAs are placed, never what
they compute: every setting must give the bits of the plain launches - on direct launches (first two calls), as a
captured and replayed call graph (later calls), inside the decimation WHILE graph (bit 1) and with the side streams of
the two-sided sweeps."""
import numpy as np
import pytest
import torch

from paper_2602_03438_b200 import workloads as W

pytestmark = pytest.mark.gpu

NAMES = ("sigma_r_L", "sigma_r_R", "GR_diag", "GR_upper", "GR_lower", "GR_corner", "GL_diag", "GL_upper", "GG_diag",
         "GG_upper", "density", "transmission", "iters_L", "iters_R")


@pytest.mark.parametrize("cfg,kw", [(1, dict(n_blocks=7, block_size=64, n_energy=6)),
                                    (1, dict(n_blocks=5, block_size=40, n_energy=3)),
                                    (2, dict(n_blocks=4, block_size=72, n_energy=2)),
                                    (3, dict(n_blocks=3, block_size=130, n_energy=2))])
def test_pdl_settings_are_bit_identical(negf_lib, cfg, kw):
    from paper_2602_03438_b200 import runner
    wl = W.make_workload(cfg, **kw)
    ref = None
    for pdl in (0, 1, 3):
        dp = runner.DevicePath(wl, want_greater=True)
        dp.ctx.set_option(negf_lib.OPT_PDL, pdl)
        got = []
        for rep in range(4):          # calls 1-2 launch directly, call 3 captures the call graphs, call 4 replays them
            dp.run_four_calls()
            torch.cuda.synchronize()
            got.append({k: dp.host(k).copy() for k in NAMES if dp.out[k].numel()})
        for rep in range(1, 4):
            for k, v in got[0].items():
                assert np.array_equal(v, got[rep][k]), (pdl, rep, k)
        if ref is None:
            ref = got[0]
            assert dp.host("status_L").tolist() == [0] * wl.n_energy
        else:
            for k, v in ref.items():
                assert np.array_equal(v, got[0][k]), (pdl, k)
        dp.ctx.close()


def test_pdl_option_range(negf_lib):
    ctx = negf_lib.Context(0)
    for v in (0, 1, 2, 3):
        ctx.set_option(negf_lib.OPT_PDL, v)
    with pytest.raises(negf_lib.NegfError):
        ctx.set_option(negf_lib.OPT_PDL, 4)
    ctx.close()
