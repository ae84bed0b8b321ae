"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times:
configs[1] complete (64 energies, n = 32, b = 64) on sampled energies against the oracle plus the
selected-block residual of Eq. 1 (SURVEY 8(c) pin P2) on EVERY energy; full block sizes of
configs[2-4] (b = 256, 1024, 2048) at reduced n / N_E against the oracle where it finishes in seconds,
else through the residual identities P2 / P3 that hold at any size."""
import numpy as np
import pytest

from oracle import assemble, pipeline
from paper_2602_03438_b200 import workloads as W
from tests.helpers import rel_fro

pytestmark = pytest.mark.gpu
TOL = 1e-10
H3_FACTOR = 3.0       # conditioning-limited chains: GPU deviation <= 3 x the oracle ensemble's own


@pytest.fixture(scope="module")
def runner_mod(negf_lib):
    from paper_2602_03438_b200 import runner
    return runner


def _gpu_boundary(dp, k):
    side = lambda t: {"sigma_r": dp.host(f"sigma_r_{t}")[k], "gamma": dp.host(f"gamma_{t}")[k],
                      "sigma_l": dp.host(f"sigma_l_{t}")[k], "sigma_g": dp.host(f"sigma_g_{t}")[k]}
    return side("L"), side("R")


def _a_blocks(wl, dp, k, sig):
    z = complex(float(wl.energies[k]), wl.eta)
    sr = pipeline._slice_sigma(sig["r"], k) if sig["r"] is not None else None
    return assemble.a_blocks(z, wl.H_diag, wl.H_upper, wl.S_diag, wl.S_upper, sr,
                             dp.host("sigma_r_L")[k], dp.host("sigma_r_R")[k])


def _residual_eq1(A, GRd, GRu, GRl):
    """max_i || sum_j A_ij G_ji - I ||_F / sqrt(b) over the block rows (P2)."""
    Ad, Au, Al = A
    n, b = Ad.shape[0], Ad.shape[1]
    worst = 0.0
    for i in range(n):
        r = Ad[i] @ GRd[i] - np.eye(b)
        if i > 0:
            r += Al[i - 1] @ GRu[i - 1]
        if i < n - 1:
            r += Au[i] @ GRl[i]
        worst = max(worst, np.linalg.norm(r) / np.sqrt(b))
    return worst


def _residual_eq2(A, B, GRd, GRu, GRl, GXd, GXu):
    """(A G^x)_ii = (Sigma^x G^A)_ii = sum_j B_ij (G^R_ij)^H over the BT pattern (P3, from Eq. 2 and
    A G^R = I), with G^x_{i+1,i} = -(G^x_{i,i+1})^H and B_{i,i-1} = -B_{i-1,i}^H; relative to the
    size of the terms."""
    Ad, Au, Al = A
    Bd, Bu = B
    n = Ad.shape[0]
    H = lambda x: np.conj(x.T)
    worst = 0.0
    for i in range(n):
        lhs = Ad[i] @ GXd[i]
        rhs = Bd[i] @ H(GRd[i])
        scale = np.linalg.norm(Ad[i]) * np.linalg.norm(GXd[i])
        if i > 0:
            lhs = lhs + Al[i - 1] @ GXu[i - 1]
            rhs = rhs - H(Bu[i - 1]) @ H(GRl[i - 1])
        if i < n - 1:
            lhs = lhs - Au[i] @ H(GXu[i])
            rhs = rhs + Bu[i] @ H(GRu[i])
        worst = max(worst, np.linalg.norm(lhs - rhs) / scale)
    return worst


def test_config1_full(runner_mod):
    wl = W.make_workload(1)
    sig = wl.sigma_s()
    dp = runner_mod.DevicePath(wl, sigma=sig)
    dp.run()
    assert int(dp.out["info_r"].abs().sum()) == 0 and int(dp.out["status_L"].abs().sum()) == 0
    GRd, GRu, GRl = dp.host("GR_diag"), dp.host("GR_upper"), dp.host("GR_lower")
    worst = max(_residual_eq1(_a_blocks(wl, dp, k, sig), GRd[k], GRu[k], GRl[k]) for k in range(wl.n_energy))
    print(f"config1 full: worst Eq.1 selected-block residual over 64 energies {worst:.2e}")
    assert worst < 1e-9
    for k in (0, 31, 63):
        s1 = {t: (None if sig[t] is None else {kk: (vv[k:k + 1] if kk != "kind" else vv) for kk, vv in sig[t].items()})
              for t in "rlg"}
        o = pipeline.solve_energy(wl, k, sigma=s1, obc_in=_gpu_boundary(dp, k), want_greater=False)
        for name, grp, key in (("GR_diag", "ret", "GR_diag"), ("GR_upper", "ret", "GR_upper"),
                               ("GR_lower", "ret", "GR_lower"), ("GL_diag", "les", "GX_diag"),
                               ("GL_upper", "les", "GX_upper")):
            assert rel_fro(dp.host(name)[k], o[grp][key]) < TOL, (k, name)
        assert abs(dp.host("transmission")[k] - o["obs"]["transmission"]) <= 1e-9 * abs(o["obs"]["transmission"]) + 1e-13


@pytest.mark.parametrize("cfg,kw,vs_oracle", [
    (2, dict(n_blocks=4, n_energy=2), True),          # b = 256, non-orthogonal S
    (3, dict(n_blocks=3, n_energy=1), True),          # b = 1024, dense BT Sigma^{R,<,>}
    (4, dict(n_blocks=3, n_energy=1), False),         # b = 2048: residual identities only
])
def test_full_block_sizes(runner_mod, cfg, kw, vs_oracle):
    wl = W.make_workload(cfg, **kw)
    sig = wl.sigma_s()
    dp = runner_mod.DevicePath(wl, want_greater=True, sigma=sig)
    dp.run()
    assert int(dp.out["info_r"].abs().sum()) == 0
    assert int(dp.out["status_L"].abs().sum()) == 0 and int(dp.out["status_R"].abs().sum()) == 0
    GRd, GRu, GRl = dp.host("GR_diag"), dp.host("GR_upper"), dp.host("GR_lower")
    for k in range(wl.n_energy):
        A = _a_blocks(wl, dp, k, sig)
        res = _residual_eq1(A, GRd[k], GRu[k], GRl[k])
        print(f"cfg{cfg} b={wl.block_size} energy {k}: Eq.1 residual {res:.2e}")
        assert res < 1e-9
        # anti-Hermiticity of the diagonal G^<> blocks (P4)
        for nm in ("GL_diag", "GG_diag"):
            g = dp.host(nm)[k]
            ah = max(np.linalg.norm(g[i] + np.conj(g[i].T)) / np.linalg.norm(g[i]) for i in range(wl.n_blocks))
            assert ah < 1e-9, (nm, ah)
        for tag, dn, un, key in (("l", "GL_diag", "GL_upper", "sigma_l"), ("g", "GG_diag", "GG_upper", "sigma_g")):
            sx = pipeline._slice_sigma(sig[tag], k) if sig[tag] is not None else None
            B = assemble.b_blocks(wl.n_blocks, wl.block_size, sx, dp.host(f"{key}_L")[k], dp.host(f"{key}_R")[k])
            r2 = _residual_eq2(A, B, GRd[k], GRu[k], GRl[k], dp.host(dn)[k], dp.host(un)[k])
            print(f"cfg{cfg} b={wl.block_size} energy {k}: Eq.2 residual ({tag}) {r2:.2e}")
            assert r2 < 1e-9
        if vs_oracle:
            s1 = {t: (None if sig[t] is None else {kk: (vv[k:k + 1] if kk != "kind" else vv) for kk, vv in sig[t].items()})
                  for t in "rlg"}
            o = pipeline.solve_energy(wl, k, sigma=s1, obc_in=_gpu_boundary(dp, k), want_greater=True)
            for name, grp, key in (("GR_diag", "ret", "GR_diag"), ("GR_upper", "ret", "GR_upper"),
                                   ("GR_lower", "ret", "GR_lower"), ("GL_diag", "les", "GX_diag"),
                                   ("GL_upper", "les", "GX_upper"), ("GG_diag", "gtr", "GX_diag"),
                                   ("GG_upper", "gtr", "GX_upper")):
                err = rel_fro(dp.host(name)[k], o[grp][key])
                assert err < TOL, (cfg, k, name, err)


def test_gemm_3m_option(runner_mod, negf_lib):
    """NEGF_OPT_GEMM_3M: 3M complex products in the compute-bound regime.  The building block stays inside
    1e-13 norm-wise, the whole path (b = 1024, dense BT Sigma) inside the 1e-10 bar against the oracle."""
    rng = np.random.default_rng(3)
    import torch
    ctx = negf_lib.Context(0)
    ctx.set_stream(torch.cuda.current_stream().cuda_stream)
    ctx.set_option(negf_lib.OPT_GEMM_3M, 1)
    m = 512
    for opA, opB in ((0, 0), (1, 0), (0, 1), (1, 1)):
        A = rng.standard_normal((8, m, m)) + 1j * rng.standard_normal((8, m, m))
        B = rng.standard_normal((8, m, m)) + 1j * rng.standard_normal((8, m, m))
        h = lambda x: np.conj(np.swapaxes(x, -1, -2))
        ref = (h(A) if opA else A) @ (h(B) if opB else B)
        dA, dB = torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda()
        dC = torch.empty_like(dA)
        ctx.zgemm_batched(opA, opB, m, m, m, 1.0, dA, m, m * m, dB, m, m * m, 0.0, None, dC, m, m * m, 8)
        err = np.linalg.norm(dC.cpu().numpy() - ref) / np.linalg.norm(ref)
        assert err < 1e-13, (opA, opB, err)
    wl = W.make_workload(3, n_blocks=3, n_energy=1)
    sig = wl.sigma_s()
    dp = runner_mod.DevicePath(wl, want_greater=True, sigma=sig)
    dp.ctx.set_option(negf_lib.OPT_GEMM_3M, 1)
    dp.run()
    assert int(dp.out["info_r"].abs().sum()) == 0
    o = pipeline.solve_energy(wl, 0, sigma=sig, obc_in=_gpu_boundary(dp, 0), want_greater=True)
    for name, grp, key in (("GR_diag", "ret", "GR_diag"), ("GR_upper", "ret", "GR_upper"), ("GL_diag", "les", "GX_diag"),
                           ("GL_upper", "les", "GX_upper"), ("GG_diag", "gtr", "GX_diag")):
        err = rel_fro(dp.host(name)[0], o[grp][key])
        print(f"3M b=1024 {name}: {err:.2e}")
        assert err < TOL, (name, err)


def test_config1_full_against_dense_definition(runner_mod):
    """The bench workload against the DEFINITION itself (dense inversion of the N = 2048 system)
    for one energy of the grid, independent of the RGF oracle."""
    from oracle import dense
    wl = W.make_workload(1)
    sig = wl.sigma_s()
    dp = runner_mod.DevicePath(wl, sigma=sig)
    dp.run()
    k = 21
    A = _a_blocks(wl, dp, k, sig)
    B = assemble.b_blocks(wl.n_blocks, wl.block_size, pipeline._slice_sigma(sig["l"], k),
                          dp.host("sigma_l_L")[k], dp.host("sigma_l_R")[k])
    d = dense.dense_green(*A, B_list=[B])
    tol = 5e-10            # the dense fp64 inverse itself carries eps * cond(A)
    assert rel_fro(dp.host("GR_diag")[k], d["GR"][0]) < tol
    assert rel_fro(dp.host("GR_upper")[k], d["GR"][1]) < tol
    assert rel_fro(dp.host("GR_lower")[k], d["GR"][2]) < tol
    assert rel_fro(dp.host("GR_corner")[k], d["GR_full"][:64, 31 * 64:]) < tol
    assert rel_fro(dp.host("GL_diag")[k], d["GX"][0][0]) < tol
    assert rel_fro(dp.host("GL_upper")[k], d["GX"][0][1]) < tol


# ---- full chain length of configs[2-4] (first / middle / last energy against the oracle) ----------
def _subset(wl, idx, sig=None):
    """The same device with the energies `idx` of its grid (Sigma_S of exactly those energies)."""
    import copy
    sub = copy.copy(wl)
    sub.energies = np.ascontiguousarray(wl.energies[idx])
    sub.weights = np.ascontiguousarray(wl.weights[idx])
    sub.name = f"{wl.name}[energies {list(idx)}]"
    if sig is None:
        parts = [wl.sigma_s(k, k + 1) for k in idx]
        sig = {t: (None if parts[0][t] is None else
                   {kk: (vv if kk == "kind" else np.concatenate([p[t][kk] for p in parts])) for kk, vv in parts[0][t].items()})
               for t in "rlg"}
    return sub, sig


def _one(sig, k):
    return {t: (None if sig[t] is None else {kk: (vv[k:k + 1] if kk != "kind" else vv) for kk, vv in sig[t].items()})
            for t in "rlg"}


_rows = []


def _compare_energy(wl, sig, dp, k, want_greater, tag, members=("mirror", "perm", "mirror+perm")):
    """All selected blocks of energy k against the oracle fed with the GPU's own boundary blocks (H2), per block,
    blocks fetched one energy at a time (the families are tens of GiB).  Bar: 1e-10 per block.  At full chain
    length the fp64 recurrences themselves are conditioning-limited at some energies (a Schur complement of a
    sub-chain is nearly singular although A is not: hazard H3, the RGF form of H2): exactly equivalent fp64
    evaluations of the oracle (mirrored chain, permuted blocks: tests/helpers.rgf_oracle_ensemble) then deviate
    from the oracle by more than 1e-10.  Such a family is labelled, never dropped, and the GPU is held to H3_FACTOR x
    the largest deviation inside the oracle's own ensemble (DESIGN.md section 5 derives the factor: the ensemble
    members invert with LAPACK's LU, K1 is a blocked Gauss-Jordan whose own bar against LAPACK is a small multiple
    of eps cond; measured ratios 0.6 ... 2.1, every row in profiles/r02_fullchain_parity.md)."""
    from tests.helpers import rgf_oracle_ensemble
    blk = lambda name: dp.out[name][k].cpu().numpy()
    side = lambda t: {"sigma_r": blk(f"sigma_r_{t}"), "gamma": blk(f"gamma_{t}"),
                      "sigma_l": blk(f"sigma_l_{t}"), "sigma_g": blk(f"sigma_g_{t}")}
    o = pipeline.solve_energy(wl, k, sigma=_one(sig, k), obc_in=(side("L"), side("R")), want_greater=want_greater)
    B_list = [o["BL"]] + ([o["BG"]] if want_greater else [])
    fams = [("GR_diag", o["ret"]["GR_diag"], lambda m: m["GR_diag"]), ("GR_upper", o["ret"]["GR_upper"], lambda m: m["GR_upper"]),
            ("GR_lower", o["ret"]["GR_lower"], lambda m: m["GR_lower"]),
            ("GL_diag", o["les"]["GX_diag"], lambda m: m["GX"][0][0]), ("GL_upper", o["les"]["GX_upper"], lambda m: m["GX"][0][1])]
    if want_greater:
        fams += [("GG_diag", o["gtr"]["GX_diag"], lambda m: m["GX"][1][0]), ("GG_upper", o["gtr"]["GX_upper"], lambda m: m["GX"][1][1])]
    per_block = lambda x, ref: np.linalg.norm(x - ref, axis=(1, 2)) / np.linalg.norm(ref, axis=(1, 2))
    gnorm = float(np.linalg.norm(o["ret"]["GR_diag"], axis=(1, 2)).max())
    anorm = float(np.linalg.norm(o["A"][0], axis=(1, 2)).max())
    errs = [float(per_block(blk(name), ref).max()) for name, ref, _ in fams]
    # each member costs one more oracle run: evaluated only when a family misses the plain bar
    ens = rgf_oracle_ensemble(o["A"], B_list, members=members, seed=k) if max(errs) > TOL else None
    bad = []
    for (name, ref, pick), e_gpu in zip(fams, errs):
        spread = max(float(per_block(pick(m), ref).max()) for m in ens) if ens is not None else float("nan")
        ok = e_gpu <= TOL or e_gpu <= H3_FACTOR * spread
        _rows.append(dict(tag=tag, k=k, E=float(wl.energies[k]), n=wl.n_blocks, b=wl.block_size, family=name, e_gpu=e_gpu,
                          spread=spread, cond_est=anorm * gnorm, label="conditioning-limited" if spread > TOL / 2 else "", ok=ok))
        if not ok:
            bad.append((name, e_gpu, spread))
    _write_fullchain_report()
    print(f"{tag} energy {k} (E = {wl.energies[k]:+.4f}), full chain n = {wl.n_blocks}: GPU vs oracle / oracle-ensemble spread: "
          + ", ".join(f"{r['family']} {r['e_gpu']:.1e}/{r['spread']:.1e}" for r in _rows[-len(fams):]))
    assert not bad, (tag, k, bad)
    c = rel_fro(blk("GR_corner"), o["ret"]["GR_corner"][0])
    gr_spread = _rows[-len(fams)]["spread"]
    assert c < max(TOL, H3_FACTOR * (gr_spread if gr_spread == gr_spread else 0.0)), (tag, k, "GR_corner", c)
    T = o["obs"]["transmission"]
    assert abs(float(dp.out["transmission"][k]) - T) <= 1e-8 * abs(T) + 1e-13


def _write_fullchain_report():
    import os
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    try:
        os.makedirs(os.path.join(root, "gpurun_out"), exist_ok=True)
        with open(os.path.join(root, "gpurun_out", "r02_fullchain_parity.md"), "w") as f:
            f.write("# Parity at full chain length, configs[2-4] (BASELINE.md section 5; SURVEY 8(c) H3)\n\n"
                    "Command: `python -m pytest tests/test_gpu_fullsize.py -m gpu -s -k 'full_chain or full_size'`\n\n"
                    "GPU err = max over the blocks of a family of the relative Frobenius error against the fp64 oracle fed "
                    "with the GPU's own boundary blocks; ensemble spread = the same measure between the oracle and exactly "
                    "equivalent fp64 evaluations of itself (mirrored chain, permuted blocks, both); cond est = max ||A_ii||_F "
                    "max ||G_ii||_F.  Rule: GPU err <= 1e-10, else GPU err <= 3x spread (the ensemble is evaluated only for "
                    "energies where some family misses the plain bar; nan = not needed).\n\n"
                    "| config | n | b | energy | E | family | GPU err | ensemble spread | cond est | label | rule |\n"
                    "|---|---|---|---|---|---|---|---|---|---|---|\n")
            for r in _rows:
                f.write(f"| {r['tag']} | {r['n']} | {r['b']} | {r['k']} | {r['E']:+.5f} | {r['family']} | {r['e_gpu']:.2e} | "
                        f"{r['spread']:.2e} | {r['cond_est']:.1e} | {r['label']} | {'ok' if r['ok'] else 'FAIL'} |\n")
    except OSError:
        pass


def test_config2_full_chain_length(runner_mod):
    """configs[2]: n = 64, b = 256, non-orthogonal S; first, middle and last energy of the 256-point grid."""
    wl, sig = _subset(W.make_workload(2), [0, 128, 255])
    dp = runner_mod.DevicePath(wl, want_greater=False, sigma=sig)
    dp.run()
    assert int(dp.out["info_r"].abs().sum()) == 0 and int(dp.out["status_L"].abs().sum() + dp.out["status_R"].abs().sum()) == 0
    try:
        for k in range(3):
            _compare_energy(wl, sig, dp, k, False, "configs[2]")
    finally:
        _release(dp)


def test_config3_full_chain_length(runner_mod):
    """configs[3]: n = 40, b = 1024, dense block-tridiagonal Sigma^{R,<,>}_S; first, middle and last energy of the grid
    (the oracle needs ~10 TFLOP per energy)."""
    wl, sig = _subset(W.make_workload(3), [0, 16, 31])
    dp = runner_mod.DevicePath(wl, want_greater=True, sigma=sig)
    dp.run()
    assert int(dp.out["info_r"].abs().sum()) == 0 and int(dp.out["status_L"].abs().sum() + dp.out["status_R"].abs().sum()) == 0
    try:
        for k in range(3):
            _compare_energy(wl, sig, dp, k, True, "configs[3]", members=("mirror",))           # one more oracle run per energy (18 s each)
    finally:
        _release(dp)


def test_config4_full_size_against_the_oracle(runner_mod):
    """configs[4] exactly as bench.py runs it (all 8 energies resident, n = 20, b = 2048, one negf_pipeline_device call);
    the middle energy against the oracle on the full chain (33 TFLOP on the host), Eq. 1 residual on the rest."""
    import torch
    wl = W.make_workload(4)
    sig = wl.sigma_s()
    dp = runner_mod.DevicePath(wl, sigma=sig)
    dp.run()
    torch.cuda.synchronize()
    for nm in ("info_r", "info_x", "status_L", "status_R"):
        assert int(dp.out[nm].abs().sum()) == 0, nm
    try:
        _compare_energy(wl, sig, dp, 3, True, "configs[4]", members=("mirror+perm",))
        for k in (0, 7):
            blk = lambda name: dp.out[name][k].cpu().numpy()
            z = complex(float(wl.energies[k]), wl.eta)
            A = assemble.a_blocks(z, wl.H_diag, wl.H_upper, None, None, None, blk("sigma_r_L"), blk("sigma_r_R"))
            res = _residual_eq1(A, blk("GR_diag"), blk("GR_upper"), blk("GR_lower"))
            print(f"configs[4] energy {k}: Eq.1 selected-block residual {res:.2e}")
            assert res < 1e-9
    finally:
        _release(dp)


def _release(dp):
    """Frees a DevicePath's tensors even when the test failed (pytest keeps the frame of a failed test alive, and the
    next full-size case needs the memory)."""
    import gc
    import torch
    dp.out.clear()
    for nm in ("workspace", "H_diag", "H_upper", "S_diag", "S_upper", "sig_dev"):
        setattr(dp, nm, None)
    dp.ctx.set_workspace(None)
    gc.collect()
    torch.cuda.empty_cache()
