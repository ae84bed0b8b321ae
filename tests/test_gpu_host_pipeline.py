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
    assert rel_fro(hp.out["GR_diag"].numpy()[k], o["ret"]["GR_diag"]) < 1e-6
    assert rel_fro(hp.out["GL_diag"].numpy()[k], o["les"]["GX_diag"]) < 1e-6
