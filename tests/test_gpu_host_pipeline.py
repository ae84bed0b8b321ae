"""negf_pipeline_host (host buffers in and out, the end-to-end call of bench.py) against the four device
calls on the same inputs, and against the oracle end to end."""
import numpy as np
import pytest

from oracle import pipeline
from paper_2602_03438_b200 import workloads as W
from tests.helpers import rel_fro

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("cfg,kw", [(0, {}), (1, dict(n_blocks=6, block_size=64, n_energy=7)),
                                    (2, dict(n_blocks=4, block_size=40, n_energy=5)),
                                    (3, dict(n_blocks=3, block_size=130, n_energy=3))])
def test_pipeline_host_matches_device_calls(negf_lib, cfg, kw):
    from paper_2602_03438_b200 import runner
    wl = W.make_workload(cfg, **kw)
    hp = runner.HostPath(wl, want_greater=True)
    up, down = hp.run()
    assert up > 0 and down > 0
    assert hp.out["info"].tolist() == [0] * wl.n_energy
    dp = runner.DevicePath(wl, want_greater=True)
    dp.run()
    for nm in ("GR_diag", "GR_upper", "GR_lower", "GL_diag", "GL_upper", "GG_diag", "GG_upper"):
        # same kernels on the same data; energy groups may change launch shapes, not the arithmetic per block
        assert rel_fro(hp.out[nm].numpy(), dp.host(nm)) < 1e-12, nm
    for nm in ("ldos", "transmission", "bond_current", "contact_current"):
        assert np.allclose(hp.out[nm].numpy(), dp.host(nm), rtol=1e-10, atol=1e-13), nm
    d = dp.host("density")
    assert np.allclose(hp.out["density"].numpy(), d, rtol=1e-10, atol=1e-12 * np.abs(d).max())
    # and against the oracle end to end (looser: the decimation's conditioning, hazard H2)
    k = wl.n_energy // 2
    o = pipeline.solve_energy(wl, k, want_greater=True)
    d_sig = max(rel_fro(dp.host(f"sigma_r_{t}")[k], o[s]["sigma_r"]) for t, s in (("L", "left"), ("R", "right")))
    assert rel_fro(hp.out["GR_diag"].numpy()[k], o["ret"]["GR_diag"]) <= 10 * d_sig + 1e-10
    assert rel_fro(hp.out["GL_diag"].numpy()[k], o["les"]["GX_diag"]) <= 10 * d_sig + 1e-10


@pytest.mark.parametrize("cfg,kw,groups", [(1, dict(n_blocks=6, block_size=24, n_energy=37), 0),     # automatic: 4 groups
                                           (1, dict(n_blocks=5, block_size=64, n_energy=7), 3),      # ragged groups 3+3+1
                                           (0, dict(n_blocks=4, block_size=16, n_energy=2), 4),      # more groups than pairs
                                           (2, dict(n_blocks=4, block_size=40, n_energy=9), 2),      # S != I
                                           (3, dict(n_blocks=3, block_size=130, n_energy=4), 2),     # BT Sigma, one-sided path
                                           (4, dict(n_blocks=3, block_size=130, n_energy=3), 0)])    # automatic: 1 group
def test_pipeline_device_equals_four_calls(negf_lib, cfg, kw, groups):
    """negf_pipeline_device (the scheduler may split the batch into concurrent energy groups on its own streams
    and workspace slices) against the four calls made one after the other: same kernels on the same data per
    energy, so the blocks are bit-identical; the density is a sum of per-group partial sums (other rounding
    order).  Twice, so that the children's cached call graphs are replayed too."""
    import torch
    from paper_2602_03438_b200 import runner
    wl = W.make_workload(cfg, **kw)
    ref = runner.DevicePath(wl, want_greater=True)
    ref.run_four_calls()
    dp = runner.DevicePath(wl, want_greater=True)
    dp.ctx.set_option(negf_lib.OPT_ENERGY_GROUPS, groups)
    names = [k for k in dp.out if k != "density"]
    for rep in range(3):
        for k in dp.out:
            dp.out[k].zero_()
        dp.run()
        torch.cuda.synchronize()
        for k in names:
            assert np.array_equal(dp.host(k), ref.host(k)), (rep, k)
        d = ref.host("density")
        assert np.allclose(dp.host("density"), d, rtol=1e-12, atol=1e-14 * np.abs(d).max())
    assert int(dp.out["info_r"].abs().sum()) == 0 and int(dp.out["status_L"].abs().sum()) == 0


def test_pipeline_device_leaves_caller_stream_ordered(negf_lib):
    """Everything the groups do is joined to the caller's stream inside the call: a copy enqueued on that
    stream right after the call sees the final outputs."""
    import torch
    from paper_2602_03438_b200 import runner
    wl = W.make_workload(1, n_blocks=6, block_size=32, n_energy=40)
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        dp = runner.DevicePath(wl, want_greater=False)
        dp.run()
        snap = dp.out["GL_diag"].clone()
        trans = dp.out["transmission"].clone()
    st.synchronize()
    ref = runner.DevicePath(wl, want_greater=False)
    ref.run_four_calls()
    torch.cuda.synchronize()
    assert np.array_equal(snap.cpu().numpy(), ref.host("GL_diag"))
    assert np.array_equal(trans.cpu().numpy(), ref.host("transmission"))
