"""Regression tests for defects found by review of round 1: a data race in the blocked inverse,
a stale cached decimation graph, first-failure semantics of `info`, and negf_pipeline_host with mixed
Sigma kinds.  All through the C ABI."""
import numpy as np
import pytest
import torch

from oracle import pipeline
from paper_2602_03438_b200 import workloads as W
from tests.helpers import rel_fro

pytestmark = pytest.mark.gpu


def _rand(rng, *shape):
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


@pytest.mark.parametrize("b,batches", [(130, (1, 5, 8)), (256, (1, 3, 8)), (1024, (1, 2, 8))])
def test_blocked_inverse_is_deterministic_under_concurrency(negf_lib, b, batches):
    """K1 above b = 96 finalises the rows above each panel in place (P' = -T Dinv, C == A): one CTA must own
    all columns of the rows it reads.  A second busy stream perturbs the CTA scheduling; every repetition
    must give the bits of the first one and agree with LAPACK."""
    rng = np.random.default_rng(b)
    busy_stream = torch.cuda.Stream()
    x = torch.randn(4096, 4096, device="cuda")
    ctx = negf_lib.Context(0)
    main = torch.cuda.current_stream()
    ctx.set_stream(main.cuda_stream)
    for batch in batches:
        A = _rand(rng, batch, b, b) / np.sqrt(b) + 0.3 * np.eye(b)
        ref = np.linalg.inv(A)
        p = negf_lib.Problem(2, b, batch, None, None, None, None, None, 0.0)
        ws = torch.empty(negf_lib.Context.workspace_bytes(p), dtype=torch.uint8, device="cuda")
        ctx.set_workspace(ws)
        hA = torch.from_numpy(A).cuda()
        info = torch.zeros(batch, dtype=torch.int32, device="cuda")
        first = None
        for rep in range(12 if b < 1024 else 5):
            dA = hA.clone()
            torch.cuda.synchronize()
            with torch.cuda.stream(busy_stream):
                for _ in range(1 + rep % 4):
                    x = (x @ x) * 1e-4
            ctx.zinverse_batched(b, dA, b * b, batch, info)
            torch.cuda.synchronize()
            got = dA.cpu().numpy()
            assert info.cpu().tolist() == [0] * batch
            if first is None:
                first = got
                for e in range(batch):
                    err = np.linalg.norm(got[e] - ref[e]) / np.linalg.norm(ref[e])
                    assert err < 50e-14 * np.linalg.cond(A[e]) + 1e-13, (batch, e, err)
            else:
                assert np.array_equal(first, got), (b, batch, rep)
    ctx.close()


def test_in_place_gemm_is_rejected_unless_one_cta_owns_the_rows(negf_lib):
    """negf_zgemm_batched with C == A and more than 16 columns would let two CTAs race on A: refused."""
    ctx = negf_lib.Context(0)
    ctx.set_stream(torch.cuda.current_stream().cuda_stream)
    a = torch.zeros(2, 64, 64, dtype=torch.complex128, device="cuda")
    bm = torch.zeros(2, 64, 64, dtype=torch.complex128, device="cuda")
    with pytest.raises(negf_lib.NegfError):
        ctx.zgemm_batched(0, 0, 64, 64, 64, 1.0, a, 64, 64 * 64, bm, 64, 64 * 64, 0.0, None, a, 64, 64 * 64, 2)
    with pytest.raises(negf_lib.NegfError):
        ctx.zgemm_batched(0, 0, 64, 64, 64, 1.0, a, 64, 64 * 64, bm, 64, 64 * 64, 0.0, None, bm, 64, 64 * 64, 2)
    ctx.close()


def test_decimation_graph_is_not_replayed_on_another_carve_up(negf_lib):
    """One context and ONE workspace buffer reused for problems with the same b and the same number of batch
    entries but another n (other scratch offsets) or another split leads x energies: the cached WHILE graph of
    the doublings must not be replayed on the old offsets."""
    from paper_2602_03438_b200 import runner
    ctx = negf_lib.Context(0)
    big = torch.empty(64 << 20, dtype=torch.uint8, device="cuda")

    def run(wl, pair, shared):
        dp = runner.DevicePath(wl, want_greater=True, ctx=ctx if shared else None)
        if shared:
            assert dp.workspace.numel() <= big.numel()
            dp.workspace = big
            dp.ctx.set_workspace(big)
        dp.obc(pair=pair)
        dp.obc(pair=pair)
        torch.cuda.synchronize()
        return {k: dp.host(k).copy() for k in dp.out if k.endswith(("_L", "_R"))}

    wl_a = W.make_workload(1, n_blocks=4, block_size=24, n_energy=4)
    wl_b = W.make_workload(1, n_blocks=7, block_size=24, n_energy=4)     # same b, same N_E, other n
    wl_c = W.make_workload(1, n_blocks=7, block_size=24, n_energy=8)
    for wl, pair in ((wl_a, True), (wl_b, True), (wl_c, False), (wl_b, True), (wl_a, True)):
        got = run(wl, pair, shared=True)
        ref = run(wl, pair, shared=False)
        assert int(got["iters_L"].min()) > 5 and got["status_L"].tolist() == [0] * wl.n_energy
        for k in ref:
            assert np.array_equal(got[k], ref[k]), (wl.name, pair, k)
    ctx.close()


def test_info_keeps_the_first_failing_block(negf_lib):
    """Two singular diagonal blocks on the chain of one energy: info names the first one met (include/negf.h),
    for the small-block kernels as for the blocked ones."""
    from paper_2602_03438_b200 import runner
    for b in (12, 40, 130):
        wl = W.make_workload(0, n_blocks=5, block_size=b, n_energy=1)
        wl.energies = np.array([0.3, 0.5]); wl.weights = np.ones(2)
        wl.eta = 0.0
        wl.H_upper[...] = 0.0                                  # decoupled blocks: A_ii = z - H_ii
        for i in (1, 3):
            wl.H_diag[i] = np.diag(np.full(b, 0.5)).astype(complex)      # singular at E = 0.5 only
        dp = runner.DevicePath(wl, want_greater=False)
        zero = torch.zeros(2, b, b, dtype=torch.complex128, device="cuda")
        sr = negf_lib.make_sigma(negf_lib.SIGMA_NONE, left=zero, right=zero)
        dp.ctx.set_option(negf_lib.OPT_GRAPH_LOOPS, 0)
        # one-sided order of elimination for b > 128; two-sided (left chain 0, 1 | right chain 4, 3) below:
        # block 1 (code 2) and block 3 (code 4) are both "first" on their chain there
        dp.ctx.rgf_retarded(dp.problem, sr, dp.out["GR_diag"], None, None, None, 0, dp.out["info_r"])
        info = dp.host("info_r").tolist()
        assert info[0] == 0
        assert info[1] == 2 if b > 128 else info[1] in (2, 4), (b, info)


def test_pipeline_host_mixed_sigma_kinds(negf_lib):
    """Scalar Sigma^R_S with block-tridiagonal Sigma^<_S / Sigma^>_S: every family is staged by its own kind."""
    from paper_2602_03438_b200 import runner
    wl = W.make_workload(3, n_blocks=4, block_size=24, n_energy=3)
    orig = wl.sigma_s

    def mixed(lo=0, hi=None):
        s = orig(lo, hi)
        ne = s["l"]["diag"].shape[0]
        s["r"] = {"kind": "scalar", "value": np.full(ne, -0.02j, dtype=np.complex128)}
        return s
    wl.sigma_s = mixed
    hp = runner.HostPath(wl, want_greater=True)
    hp.run()
    assert hp.out["info"].tolist() == [0] * wl.n_energy
    dp = runner.DevicePath(wl, want_greater=True)
    dp.run()
    torch.cuda.synchronize()
    for nm in ("GR_diag", "GR_upper", "GL_diag", "GL_upper", "GG_diag", "GG_upper"):
        assert rel_fro(hp.out[nm].numpy(), dp.host(nm)) < 1e-12, nm
    k = 1
    side = lambda t: {"sigma_r": dp.host(f"sigma_r_{t}")[k], "gamma": dp.host(f"gamma_{t}")[k],
                      "sigma_l": dp.host(f"sigma_l_{t}")[k], "sigma_g": dp.host(f"sigma_g_{t}")[k]}
    o = pipeline.solve_energy(wl, k, sigma=mixed(k, k + 1), obc_in=(side("L"), side("R")), want_greater=True)
    assert rel_fro(hp.out["GR_diag"].numpy()[k], o["ret"]["GR_diag"]) < 1e-10
    assert rel_fro(hp.out["GL_upper"].numpy()[k], o["les"]["GX_upper"]) < 1e-10
    assert rel_fro(hp.out["GG_diag"].numpy()[k], o["gtr"]["GX_diag"]) < 1e-10


def test_pipeline_host_restores_the_callers_workspace(negf_lib):
    """A negf_pipeline_host that fails AFTER it switched to its staging workspace (max_iter = 0 is refused by
    the decimation call inside it) leaves the context on the caller's workspace."""
    from paper_2602_03438_b200 import runner
    wl = W.make_workload(1, n_blocks=4, block_size=24, n_energy=3)
    dp = runner.DevicePath(wl, want_greater=False)
    dp.run()
    ref = dp.host("GL_diag").copy()
    hp = runner.HostPath(wl, ctx=dp.ctx, want_greater=False)
    wl.max_iter = 0
    with pytest.raises(negf_lib.NegfError):
        hp.run()
    wl.max_iter = 64
    dp.out["GL_diag"].zero_()
    dp.run()                                   # same context, its own workspace still set
    torch.cuda.synchronize()
    assert np.array_equal(dp.host("GL_diag"), ref)
