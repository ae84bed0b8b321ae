"""negf_zinverse_batched_static (include/negf.h): the no-allocation variant of the batched inverse K1, whose scratch is
a file-scope `static __device__` array of the library instead of the caller's workspace.  Checked against the existing
path (negf_zinverse_batched with a torch-owned workspace) on two calls in a row: the second call finds the first
call's contents in the shared array and must not depend on them.  Collected last on purpose (the suite runs with
`pytest -x`); passes alone in a fresh process and after the other GPU tests."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _inputs(seed, batch, b):
    rng = np.random.default_rng(seed)
    A = (rng.standard_normal((batch, b, b)) + 1j * rng.standard_normal((batch, b, b))) / np.sqrt(b) + 0.3 * np.eye(b)
    A[0, 0, :] *= 1e-3                      # row pivoting on the first column
    return A


@pytest.mark.parametrize("b,batch", [(130, 5), (256, 3), (515, 2), (64, 7)])
def test_static_scratch_inverse_matches_workspace_path(negf_lib, b, batch):
    import torch
    c = negf_lib.Context(0)
    c.set_stream(torch.cuda.current_stream().cuda_stream)
    p = negf_lib.Problem(2, b, batch, None, None, None, None, None, 0.0)
    ws = torch.empty(negf_lib.Context.workspace_bytes(p), dtype=torch.uint8, device="cuda")
    for call, (seed, nb) in enumerate(((11 * b, batch), (13 * b + 1, max(1, batch - 1)))):   # two calls in a row
        A = _inputs(seed, nb, b)
        ref = np.linalg.inv(A)
        # existing path: caller-owned workspace
        d_ws = torch.from_numpy(A).cuda()
        info_ws = torch.full((nb,), -7, dtype=torch.int32, device="cuda")
        c.set_workspace(ws)
        c.zinverse_batched(b, d_ws, b * b, nb, info_ws)
        # new path: no workspace attached at all, scratch inside the library
        c.set_workspace(None)
        d_st = torch.from_numpy(A).cuda()
        info_st = torch.full((nb,), -7, dtype=torch.int32, device="cuda")
        free0 = torch.cuda.mem_get_info()[0]
        c.zinverse_batched_static(b, d_st, b * b, nb, info_st)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free0, "the no-allocation entry point changed the free device memory"
        assert info_ws.cpu().tolist() == [0] * nb and info_st.cpu().tolist() == [0] * nb
        got_ws, got_st = d_ws.cpu().numpy(), d_st.cpu().numpy()
        for e in range(nb):
            # the tolerance of tests/test_gpu_blocks.py::test_zinverse_batched (K1 bar) ...
            cond = np.linalg.cond(A[e])
            err = np.linalg.norm(got_st[e] - ref[e]) / np.linalg.norm(ref[e])
            assert err < 1e-14 * cond * 50 + 1e-13, (call, e, err, cond)
            # ... and against the existing path: same kernels in the same order
            dev = np.linalg.norm(got_st[e] - got_ws[e]) / np.linalg.norm(got_ws[e])
            assert dev < 1e-14 * cond * 50 + 1e-13, (call, e, dev)
    c.close()


def test_static_scratch_limit_is_reported(negf_lib):
    """Beyond NEGF_STATIC_SCRATCH_BYTES the call returns NEGF_ESTATICLIMIT with a clear message and launches nothing."""
    import torch
    c = negf_lib.Context(0)
    c.set_stream(torch.cuda.current_stream().cuda_stream)
    b, batch = 256, 64
    A = torch.eye(b, dtype=torch.complex128, device="cuda").repeat(batch, 1, 1).contiguous()
    before = A.clone()
    n0 = c.launch_count()
    with pytest.raises(negf_lib.NegfError, match="static scratch"):
        c.zinverse_batched_static(b, A, b * b, batch, None)
    torch.cuda.synchronize()
    assert c.launch_count() == n0 and torch.equal(A, before)
    assert negf_lib.strerror(negf_lib.ESTATICLIMIT).startswith("problem exceeds the static scratch")
    c.close()
