"""Pins for the oracle's own FFT (oracle/gpe_oracle.c: dft_direct, fft_radix2, fft2_grid).

Pinned against things other than itself: numpy's pocketfft (an independent library routine),
the DFT definition written as a dense matrix product, and the textbook identities (impulse,
shift theorem, Parseval, round trip).  SURVEY.md 8(c) "What pins each part", row FFT."""
import numpy as np
import pytest

from oracle import gpe_oracle as O


def _rand(shape, seed):
    rng = np.random.default_rng(seed)
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


@pytest.mark.parametrize("n", [2, 4, 8, 16, 32, 64, 128, 1024])
def test_fft1_matches_dft_matrix_and_numpy(n):
    a = _rand(n, n)
    j = np.arange(n)
    F = np.exp(-2j * np.pi * np.outer(j, j) / n)          # the definition, e^{-ikx} kernel
    got = O.fft1(a, -1)
    assert np.max(np.abs(got - F @ a)) <= 1e-12 * n
    assert np.max(np.abs(got - np.fft.fft(a))) <= 1e-12 * n
    inv = O.fft1(a, +1)                                     # 1-D inverse is unnormalised
    assert np.max(np.abs(inv - np.conj(F) @ a)) <= 1e-12 * n


def test_radix2_equals_direct_at_64():
    a = _rand(64, 5)
    assert np.max(np.abs(O.fft1(a, -1) - O.fft1(a, -1, force_direct=True))) <= 1e-12


@pytest.mark.parametrize("shape", [(8, 8), (16, 64), (64, 32), (128, 256)])
def test_fft2_matches_numpy_and_roundtrip(shape):
    a = _rand(shape, 11)
    f = O.fft2(a, -1)
    assert np.max(np.abs(f - np.fft.fft2(a))) <= 1e-11 * np.sqrt(a.size)
    back = O.fft2(f, +1)                                    # carries 1/(nx*ny)
    assert np.max(np.abs(back - a)) <= 1e-13 * np.sqrt(a.size)
    inv = O.fft2(a, +1)
    assert np.max(np.abs(inv - np.fft.ifft2(a))) <= 1e-13


def test_impulse_shift_parseval():
    nx, ny = 64, 128
    imp = np.zeros((nx, ny), complex)
    imp[0, 0] = 1.0
    assert np.max(np.abs(O.fft2(imp) - 1.0)) <= 1e-14      # impulse -> constant
    sx, sy = 5, 9
    imp2 = np.zeros((nx, ny), complex)
    imp2[sx, sy] = 1.0
    p = np.arange(nx)[:, None]
    q = np.arange(ny)[None, :]
    expect = np.exp(-2j * np.pi * (p * sx / nx + q * sy / ny))   # shift theorem, sign pin
    assert np.max(np.abs(O.fft2(imp2) - expect)) <= 1e-12
    a = _rand((nx, ny), 3)
    f = O.fft2(a)
    assert abs(np.sum(np.abs(f) ** 2) / (nx * ny) - np.sum(np.abs(a) ** 2)) <= 1e-9  # Parseval


def test_axes_not_transposed():
    # a plane wave along x only must land at (p, 0), not (0, p)
    nx, ny = 32, 64
    x = np.arange(nx)[:, None] * np.ones((1, ny))
    a = np.exp(2j * np.pi * 3 * x / nx)
    f = O.fft2(a)
    assert abs(f[3, 0] - nx * ny) <= 1e-9
    f[3, 0] = 0
    assert np.max(np.abs(f)) <= 1e-9


@pytest.mark.parametrize("n", [96, 160, 240, 90, 250])
def test_non_power_of_two_lengths_take_the_definition(n):
    """SURVEY.md 8(f) f4 ("non-optimal grid sizes"): lengths that are not powers of two go
    through dft_direct.  Pinned against the DFT matrix and numpy, both directions."""
    a = _rand(n, n)
    j = np.arange(n)
    F = np.exp(-2j * np.pi * np.outer(j, j) / n)
    got = O.fft1(a, -1)
    assert np.max(np.abs(got - F @ a)) <= 1e-12 * n
    assert np.max(np.abs(got - np.fft.fft(a))) <= 1e-12 * n
    assert np.max(np.abs(O.fft1(a, +1) - np.conj(F) @ a)) <= 1e-12 * n


@pytest.mark.parametrize("shape", [(96, 160), (240, 64), (128, 90)])
def test_fft2_non_power_of_two(shape):
    a = _rand(shape, 17)
    f = O.fft2(a, -1)
    assert np.max(np.abs(f - np.fft.fft2(a))) <= 1e-11 * np.sqrt(a.size)
    assert np.max(np.abs(O.fft2(f, +1) - a)) <= 1e-13 * np.sqrt(a.size)
