"""Pins of the oracle's DFT / FFT (SURVEY.md 8(c) table, row "FFT").

Independent references: the DFT sum written with numpy matrix algebra, numpy.fft
(a different library routine than the oracle's own radix-2), and closed forms
(delta <-> constant, plane wave <-> single bin, Parseval).
"""
import numpy as np
import pytest

import oracle as orc


def _rand(n, seed):
    r = np.random.default_rng(seed)
    return r.standard_normal(n) + 1j * r.standard_normal(n)


@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 8, 16, 32, 64])
def test_naive_dft_is_the_definition(n):
    a = _rand(n, n)
    j = np.arange(n)
    F = np.exp(-2j * np.pi * np.outer(j, j) / n)  # X_m = sum_j x_j e^{-2 pi i jm/N}
    np.testing.assert_allclose(orc.dft_naive(a, -1), F @ a, rtol=0, atol=1e-13 * n)
    np.testing.assert_allclose(orc.dft_naive(a, +1), F.conj() @ a, rtol=0, atol=1e-13 * n)


@pytest.mark.parametrize("n", [2, 4, 8, 16, 32, 64, 256, 2048])
def test_radix2_equals_naive_and_numpy(n):
    a = _rand(n, 100 + n)
    got = orc.fft_radix2(a, -1)
    scale = np.abs(got).max()
    if n <= 64:
        np.testing.assert_allclose(got, orc.dft_naive(a, -1), rtol=0, atol=1e-13 * scale)
    np.testing.assert_allclose(got, np.fft.fft(a), rtol=0, atol=1e-13 * scale)
    inv = orc.fft_radix2(a, +1)
    np.testing.assert_allclose(inv, np.fft.ifft(a) * n, rtol=0, atol=1e-13 * scale)


@pytest.mark.parametrize("n", [8, 64, 1024])
def test_radix2_inverse_of_forward(n):
    a = _rand(n, 7)
    back = orc.fft_radix2(orc.fft_radix2(a, -1), +1) / n
    np.testing.assert_allclose(back, a, rtol=0, atol=1e-13)


def test_delta_constant_planewave_parseval():
    n = 128
    d = np.zeros(n, complex)
    d[0] = 1.0
    np.testing.assert_allclose(orc.fft_radix2(d, -1), np.ones(n), atol=1e-14)
    np.testing.assert_allclose(orc.fft_radix2(np.ones(n, complex), -1), n * d, atol=1e-12)
    m = 37
    pw = np.exp(2j * np.pi * m * np.arange(n) / n)
    e = np.zeros(n, complex)
    e[m] = n
    np.testing.assert_allclose(orc.fft_radix2(pw, -1), e, atol=1e-11)
    # a delta at j0 gives e^{-2 pi i j0 m / n}: fixes the SIGN of the forward transform
    d2 = np.zeros(n, complex)
    d2[3] = 1.0
    np.testing.assert_allclose(orc.fft_radix2(d2, -1), np.exp(-2j * np.pi * 3 * np.arange(n) / n), atol=1e-13)
    a = _rand(n, 3)
    assert abs(np.sum(np.abs(orc.fft_radix2(a, -1)) ** 2) / n - np.sum(np.abs(a) ** 2)) < 1e-11


@pytest.mark.parametrize("ny,nx,naive_max", [(4, 4, 32), (8, 16, 32), (16, 8, 0), (64, 32, 32), (32, 128, 0),
                                             (64, 64, 16)])
def test_fft2_against_numpy_fft2(ny, nx, naive_max):
    """2-D transform of both components, rows then columns, rectangular grids, both code paths."""
    r = np.random.default_rng(ny * 1000 + nx)
    psi = r.standard_normal((ny, nx, 2)) + 1j * r.standard_normal((ny, nx, 2))
    p = orc.params(nx, ny, 1.0, 1.0, naive_max=naive_max)
    fwd = orc.fft2(psi, p, -1)
    ref = np.fft.fft2(psi, axes=(0, 1))
    np.testing.assert_allclose(fwd, ref, rtol=0, atol=1e-13 * np.abs(ref).max())
    inv = orc.fft2(psi, p, +1)
    np.testing.assert_allclose(inv, np.fft.ifft2(psi, axes=(0, 1)), rtol=0, atol=1e-14)
    np.testing.assert_allclose(orc.fft2(fwd, p, +1), psi, rtol=0, atol=1e-13)


def test_fft2_planewave_lands_in_one_bin_and_axes_are_not_swapped():
    ny, nx = 32, 64
    my, mx = 5, 50
    y = np.arange(ny)[:, None]
    x = np.arange(nx)[None, :]
    pw = np.exp(2j * np.pi * (mx * x / nx + my * y / ny))
    psi = np.stack([pw, 2.0 * pw.conj()], axis=-1)
    out = orc.fft2(psi, orc.params(nx, ny, 1.0, 1.0, naive_max=0), -1)
    ref = np.zeros((ny, nx, 2), complex)
    ref[my, mx, 0] = nx * ny
    ref[(-my) % ny, (-mx) % nx, 1] = 2.0 * nx * ny
    np.testing.assert_allclose(out, ref, atol=1e-9)


def test_grids():
    k = orc.kgrid(8, 2 * np.pi)
    np.testing.assert_allclose(k, [0, 1, 2, 3, -4, -3, -2, -1], atol=1e-15)  # Nyquist -> -pi/dx
    np.testing.assert_allclose(orc.kgrid(64, 16.0), 2 * np.pi * np.fft.fftfreq(64, d=16.0 / 64), atol=1e-13)
    x = orc.xgrid(8, 16.0)
    np.testing.assert_allclose(x, [-8, -6, -4, -2, 0, 2, 4, 6], atol=1e-15)  # box [-L/2, L/2)
    # dk = pi / x_max
    assert abs((k[1] - k[0]) - np.pi / np.pi) < 1e-15
