"""negf_energy_convolve (Eq. 3) against the oracle's written-out sums: sizes that span several
CTA tiles with a ragged tail, both modes, conjugate / block-transposed second operand, and G^< (x) G^> of a
real run (the polarisation-like correlation of SURVEY 8(f) item 3)."""
import numpy as np
import pytest
import torch

from oracle import convolution as C
from paper_2602_03438_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _run(negf_lib, X1, X2, **kw):
    ctx = negf_lib.Context(0)
    ctx.set_stream(torch.cuda.current_stream().cuda_stream)
    ne, M = X1.shape
    d1, d2 = torch.from_numpy(X1).cuda(), torch.from_numpy(np.ascontiguousarray(X2)).cuda()
    Y = torch.empty(2 * ne - 1, M, dtype=torch.complex128, device="cuda")
    ctx.energy_convolve(ne, M, d1, d2, Y, **kw)
    return Y.cpu().numpy()


@pytest.mark.parametrize("ne,M", [(1, 5), (2, 70), (7, 1000), (64, 700), (65, 129), (200, 50), (1024, 9)])
@pytest.mark.parametrize("mode,conj2", [(0, False), (1, True)])
def test_convolution_matches_definition(negf_lib, ne, M, mode, conj2):
    rng = np.random.default_rng(ne * 7 + M + mode)
    X1 = rng.standard_normal((ne, M)) + 1j * rng.standard_normal((ne, M))
    X2 = rng.standard_normal((ne, M)) + 1j * rng.standard_normal((ne, M))
    if ne > 300:       # the O(N_E^2) definition is slow: check sampled elements
        cols = np.array([0, M // 2, M - 1])
        ref = C.energy_convolve(X1[:, cols], X2[:, cols], mode=mode, conj2=conj2, scale=0.3 - 0.2j)
        got = _run(negf_lib, X1, X2, mode=mode, conj2=conj2, scale=0.3 - 0.2j)[:, cols]
    else:
        ref = C.energy_convolve(X1, X2, mode=mode, conj2=conj2, scale=0.3 - 0.2j)
        got = _run(negf_lib, X1, X2, mode=mode, conj2=conj2, scale=0.3 - 0.2j)
    # FFT rounding: eps * log2(L) relative to the largest term of a sum
    assert np.abs(got - ref).max() <= 1e-13 * np.abs(ref).max()


def test_block_transpose_and_errors(negf_lib):
    rng = np.random.default_rng(5)
    ne, nb, b = 6, 9, 12
    X1 = rng.standard_normal((ne, nb * b * b)) + 1j * rng.standard_normal((ne, nb * b * b))
    X2 = rng.standard_normal((ne, nb * b * b)) + 1j * rng.standard_normal((ne, nb * b * b))
    ref = C.energy_convolve(X1, X2, mode=1, conj2=False, transpose_block=b)
    got = _run(negf_lib, X1, X2, mode=1, transpose_block=b)
    assert np.abs(got - ref).max() <= 1e-13 * np.abs(ref).max()
    ctx = negf_lib.Context(0)
    d = torch.zeros(4, 10, dtype=torch.complex128, device="cuda")
    y = torch.zeros(7, 10, dtype=torch.complex128, device="cuda")
    one = negf_lib.c128(1.0, 0.0)
    assert negf_lib.lib.negf_energy_convolve(ctx._h, 4, 10, 3, d.data_ptr(), d.data_ptr(), 0, 0, one, y.data_ptr()) == negf_lib.EINVAL
    assert negf_lib.lib.negf_energy_convolve(ctx._h, 4000, 10, 0, d.data_ptr(), d.data_ptr(), 0, 0, one, y.data_ptr()) == negf_lib.EUNSUPPORTED


def test_lesser_greater_correlation_of_a_run(negf_lib):
    """P^<-like quantity from a real run: sum_E G^<_ij(E) G^>_ji(E - w) on the diagonal blocks, GPU FFT route
    against the oracle's direct sums on the GPU's own G^<, G^> (identical inputs)."""
    from paper_2602_03438_b200 import runner
    wl = W.make_workload(1, n_blocks=4, block_size=16, n_energy=24)
    dp = runner.DevicePath(wl, want_greater=True)
    dp.run()
    ne, M = wl.n_energy, wl.n_blocks * 16 * 16
    GL, GG = dp.out["GL_diag"].reshape(ne, M), dp.out["GG_diag"].reshape(ne, M)
    Y = torch.empty(2 * ne - 1, M, dtype=torch.complex128, device="cuda")
    de = float(wl.energies[1] - wl.energies[0])
    scale = -1j * de / (2 * np.pi)
    dp.ctx.energy_convolve(ne, M, GL, GG, Y, mode=1, conj2=False, scale=scale, transpose_block=16)
    ref = C.energy_convolve(GL.cpu().numpy(), GG.cpu().numpy(), mode=1, scale=scale, transpose_block=16)
    assert np.abs(Y.cpu().numpy() - ref).max() <= 1e-13 * np.abs(ref).max()
