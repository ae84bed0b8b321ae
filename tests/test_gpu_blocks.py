"""K1/K2 building blocks through the C ABI against library routines (numpy matmul / LAPACK inv).
Sizes span several tiles and ragged tails."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx(negf_lib):
    import torch
    c = negf_lib.Context(0)
    c.set_stream(torch.cuda.current_stream().cuda_stream)
    return c


def _rand(rng, *shape):
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


@pytest.mark.parametrize("m,n,k", [(1, 1, 1), (8, 8, 4), (16, 16, 16), (64, 64, 64), (37, 53, 29),
                                   (128, 64, 16), (200, 130, 75), (256, 256, 256), (300, 257, 33)])
@pytest.mark.parametrize("opA,opB", [(0, 0), (1, 0), (0, 1), (1, 1)])
def test_zgemm_batched(ctx, m, n, k, opA, opB):
    import torch
    rng = np.random.default_rng(m * 1000 + n * 10 + k + opA * 2 + opB)
    batch = 3
    A = _rand(rng, batch, *((k, m) if opA else (m, k)))
    B = _rand(rng, batch, *((n, k) if opB else (k, n)))
    D = _rand(rng, batch, m, n)
    alpha, beta = 0.7 - 0.3j, -1.1 + 0.4j
    opa = (lambda x: np.conj(np.swapaxes(x, -1, -2))) if opA else (lambda x: x)
    opb = (lambda x: np.conj(np.swapaxes(x, -1, -2))) if opB else (lambda x: x)
    ref = alpha * (opa(A) @ opb(B)) + beta * D
    dA, dB, dD = (torch.from_numpy(x).cuda() for x in (A, B, D))
    dC = torch.empty_like(dD)
    ctx.zgemm_batched(opA, opB, m, n, k, alpha, dA, A.shape[2], A.shape[1] * A.shape[2], dB, B.shape[2],
                      B.shape[1] * B.shape[2], beta, dD, dC, n, m * n, batch)
    got = dC.cpu().numpy()
    err = np.linalg.norm(got - ref) / np.linalg.norm(ref)
    assert err < 1e-13, err
    # shared operand (stride 0), no addend, in-place addend
    dC2 = dD.clone()
    ctx.zgemm_batched(opA, opB, m, n, k, 1.0, dA, A.shape[2], 0, dB, B.shape[2], B.shape[1] * B.shape[2],
                      1.0, dC2, dC2, n, m * n, batch)
    ref2 = opa(A[:1]) @ opb(B) + D
    assert np.linalg.norm(dC2.cpu().numpy() - ref2) / np.linalg.norm(ref2) < 1e-13


@pytest.mark.parametrize("m,n,k,batch", [(200, 130, 75, 40), (129, 65, 17, 150), (300, 257, 33, 20), (70, 640, 130, 30),
                                         (1030, 1000, 70, 2)])
@pytest.mark.parametrize("opA,opB", [(0, 0), (1, 0), (0, 1), (1, 1)])
def test_zgemm_compute_bound_tiles(ctx, m, n, k, batch, opA, opB):
    """Launches with at least two 64 x 64 tiles per SM take the compute-bound tile configuration of K2 (two co-resident CTAs
    of 8 warps per SM, addend tile prefetched into L2): ragged rows, columns and k, every operand orientation, with an
    in-place addend (C == D), against NumPy at the K2 bar."""
    import torch
    assert ((m + 63) // 64) * ((n + 63) // 64) * batch >= 2 * 148
    rng = np.random.default_rng(m * 7 + n * 3 + k + opA * 2 + opB)
    A = _rand(rng, batch, *((k, m) if opA else (m, k)))
    B = _rand(rng, batch, *((n, k) if opB else (k, n)))
    D = _rand(rng, batch, m, n)
    alpha, beta = -0.9 + 0.2j, 1.0
    opa = (lambda x: np.conj(np.swapaxes(x, -1, -2))) if opA else (lambda x: x)
    opb = (lambda x: np.conj(np.swapaxes(x, -1, -2))) if opB else (lambda x: x)
    ref = alpha * (opa(A) @ opb(B)) + beta * D
    dA, dB, dC = (torch.from_numpy(x).cuda() for x in (A, B, D))
    ctx.zgemm_batched(opA, opB, m, n, k, alpha, dA, A.shape[2], A.shape[1] * A.shape[2], dB, B.shape[2],
                      B.shape[1] * B.shape[2], beta, dC, dC, n, m * n, batch)
    got = dC.cpu().numpy()
    for e in (0, batch // 2, batch - 1):
        assert np.linalg.norm(got[e] - ref[e]) / np.linalg.norm(ref[e]) < 1e-13, e
    assert np.linalg.norm(got - ref) / np.linalg.norm(ref) < 1e-13


@pytest.mark.parametrize("b", [1, 2, 7, 16, 33, 64, 96, 97, 130, 256, 300, 515, 1100, 2100])
def test_zinverse_batched(ctx, negf_lib, b):
    """2100 > 2048 rows: the first panels take the shared-memory cluster panel kernel instead of the register one."""
    import torch
    rng = np.random.default_rng(b)
    batch = 3 if b < 400 else 2
    A = _rand(rng, batch, b, b) / np.sqrt(b) + 0.3 * np.eye(b)
    A[0, 0, :] *= 1e-3      # force row pivoting on the first column
    if b > 2:
        A[1, :, 1] = A[1, :, 0] * (1 + 1e-9) + 1e-7 * A[1, :, 1]   # nearly dependent columns
    ref = np.linalg.inv(A)
    dA = torch.from_numpy(A).cuda()
    info = torch.full((batch,), -7, dtype=torch.int32, device="cuda")
    p = negf_lib.Problem(2, b, batch, None, None, None, None, None, 0.0)
    ws = torch.empty(negf_lib.Context.workspace_bytes(p), dtype=torch.uint8, device="cuda")
    ctx.set_workspace(ws)
    ctx.zinverse_batched(b, dA, b * b, batch, info)
    got = dA.cpu().numpy()
    assert info.cpu().tolist() == [0] * batch
    for e in range(batch):
        cond = np.linalg.cond(A[e])
        err = np.linalg.norm(got[e] - ref[e]) / np.linalg.norm(ref[e])
        assert err < 1e-14 * cond * 50 + 1e-13, (e, err, cond)
        res = np.linalg.norm(A[e] @ got[e] - np.eye(b)) / np.sqrt(b)
        assert res < 1e-14 * cond * 50 + 1e-12


def test_zinverse_singular_reports_info(ctx, negf_lib):
    import torch
    b = 40
    A = np.eye(b, dtype=complex)[None].repeat(2, 0)
    A[1, :, 5] = 0.0
    dA = torch.from_numpy(A).cuda()
    info = torch.zeros(2, dtype=torch.int32, device="cuda")
    ctx.zinverse_batched(b, dA, b * b, 2, info)
    assert info.cpu().tolist() == [0, 6]


@pytest.mark.parametrize("b", [9, 12, 17, 24, 31, 32, 33, 40, 47, 56, 63, 64])
def test_zinverse_tensor_and_register_kernels(negf_lib, b):
    """16 < b <= 64 has two K1 kernels (below, both options run the register kernel): the blocked one with rank-4 DMMA updates (NEGF_OPT_INV_TENSOR = 1, default) and the
    register-resident unblocked one (0).  Both against LAPACK at the K1 bar; sizes cover both paddings (32 and 64 rows),
    ragged last panels (b not a multiple of 4) and last tiles; the batch holds a matrix that needs pivoting at once, one
    with nearly dependent columns and ill-conditioned ones (cond up to ~1e8), where the blocked kernel must stay
    within a small factor of the unblocked one (the order of its updates is that of the unblocked elimination)."""
    import torch
    rng = np.random.default_rng(1000 + b)
    batch = 6
    A = _rand(rng, batch, b, b) / np.sqrt(b) + 0.3 * np.eye(b)
    A[0, 0, :] *= 1e-3
    A[1, :, 1] = A[1, :, 0] * (1 + 1e-9) + 1e-7 * A[1, :, 1]
    for e, c in ((3, 1e4), (4, 1e6), (5, 1e8)):                    # graded singular values
        u, _, vh = np.linalg.svd(_rand(rng, b, b))
        A[e] = (u * np.logspace(0, -np.log10(c), b)) @ vh
    ref = np.linalg.inv(A)
    errs = {}
    for opt in (1, 0):
        c = negf_lib.Context(0)
        c.set_stream(torch.cuda.current_stream().cuda_stream)
        c.set_option(negf_lib.OPT_INV_TENSOR, opt)
        dA = torch.from_numpy(A).cuda()
        info = torch.full((batch,), -7, dtype=torch.int32, device="cuda")
        c.zinverse_batched(b, dA, b * b, batch, info)
        got = dA.cpu().numpy()
        assert info.cpu().tolist() == [0] * batch
        errs[opt] = [np.linalg.norm(got[e] - ref[e]) / np.linalg.norm(ref[e]) for e in range(batch)]
        for e in range(batch):
            cond = np.linalg.cond(A[e])
            assert errs[opt][e] < 1e-14 * cond * 50 + 1e-13, (opt, e, errs[opt][e], cond)
        c.close()
    for e in range(batch):
        assert errs[1][e] <= 8 * errs[0][e] + 1e-14, (e, errs[1][e], errs[0][e])


@pytest.mark.parametrize("opt", [0, 1])
@pytest.mark.parametrize("b,col", [(12, 0), (33, 32), (64, 63), (50, 17)])
def test_zinverse_singular_both_kernels(negf_lib, opt, b, col):
    """A zero column is reported as its 1-based index by either kernel; the other entries of the batch are untouched by it."""
    import torch
    c = negf_lib.Context(0)
    c.set_stream(torch.cuda.current_stream().cuda_stream)
    c.set_option(negf_lib.OPT_INV_TENSOR, opt)
    rng = np.random.default_rng(b + col)
    A = _rand(rng, 3, b, b) / np.sqrt(b) + 0.5 * np.eye(b)
    A[1, :, col] = 0.0
    ref0, ref2 = np.linalg.inv(A[0]), np.linalg.inv(A[2])
    dA = torch.from_numpy(A).cuda()
    info = torch.zeros(3, dtype=torch.int32, device="cuda")
    c.zinverse_batched(b, dA, b * b, 3, info)
    got = dA.cpu().numpy()
    assert info.cpu().tolist() == [0, col + 1, 0]
    assert np.linalg.norm(got[0] - ref0) / np.linalg.norm(ref0) < 1e-11
    assert np.linalg.norm(got[2] - ref2) / np.linalg.norm(ref2) < 1e-11
    c.close()
