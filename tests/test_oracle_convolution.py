"""Pins of the Eq. 3 oracle (oracle/convolution.py): closed forms and an independent route."""
import numpy as np

from oracle import convolution as C


def test_delta_shifts():
    rng = np.random.default_rng(0)
    ne, M, k0 = 7, 5, 3
    X1 = rng.standard_normal((ne, M)) + 1j * rng.standard_normal((ne, M))
    d = np.zeros((ne, M), complex); d[k0] = 1.0
    Y = C.energy_convolve(X1, d)
    assert np.allclose(Y[k0:k0 + ne], X1) and np.allclose(Y[:k0], 0) and np.allclose(Y[k0 + ne:], 0)
    Yc = C.energy_convolve(X1, d, mode=1)           # lag l = k1 - k0 at index l + ne - 1
    for k1 in range(ne):
        assert np.allclose(Yc[k1 - k0 + ne - 1], X1[k1])


def test_polynomial_product_binomial():
    # (1 + x)^3 * (1 + x)^3 = (1 + x)^6: coefficients are binomials
    a = np.array([1, 3, 3, 1], complex)[:, None]
    Y = C.energy_convolve(a, a)
    assert np.allclose(Y[:, 0], [1, 6, 15, 20, 15, 6, 1])


def test_against_library_convolve_and_fft_route():
    rng = np.random.default_rng(1)
    ne, M = 9, 6
    X1 = rng.standard_normal((ne, M)) + 1j * rng.standard_normal((ne, M))
    X2 = rng.standard_normal((ne, M)) + 1j * rng.standard_normal((ne, M))
    Y = C.energy_convolve(X1, X2, conj2=True, scale=0.5 - 2j)
    for e in range(M):
        assert np.allclose(Y[:, e], (0.5 - 2j) * np.convolve(X1[:, e], np.conj(X2[:, e])))
    L = 32
    F = np.fft.ifft(np.fft.fft(X1, L, axis=0) * np.fft.fft(np.conj(X2), L, axis=0), axis=0)[:2 * ne - 1]
    assert np.allclose(Y, (0.5 - 2j) * F)
    # correlation = convolution with the second operand reversed in energy
    Yc = C.energy_convolve(X1, X2, mode=1)
    assert np.allclose(Yc, C.energy_convolve(X1, X2[::-1]))


def test_block_transpose_of_second_operand():
    rng = np.random.default_rng(2)
    ne, nb, b = 3, 2, 3
    X1 = rng.standard_normal((ne, nb * b * b)) + 0j
    X2 = rng.standard_normal((ne, nb, b, b)) + 1j * rng.standard_normal((ne, nb, b, b))
    Y = C.energy_convolve(X1, X2.reshape(ne, -1), transpose_block=b)
    Yt = C.energy_convolve(X1, np.swapaxes(X2, -1, -2).reshape(ne, -1))
    assert np.allclose(Y, Yt)
