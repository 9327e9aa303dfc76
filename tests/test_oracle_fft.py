"""Pins for the oracle's own FFT (oracle/cwo_oracle.c) against the DFT definition.

Conventions under test: forward kernel exp(-i 2 pi j k / n), inverse
exp(+...) with 1/n.  Every check compares with something that is not the radix-2 recursion:
the O(n^2) definition, closed forms, or invariants.
"""
import numpy as np
import pytest

from conftest import rel_l2


def _rand(shape, seed):
    r = np.random.default_rng(seed)
    return r.standard_normal(shape) + 1j * r.standard_normal(shape)


@pytest.mark.parametrize("n", [1, 2, 4, 8, 16, 32, 64])
@pytest.mark.parametrize("sign", [-1, +1])
def test_fft1d_equals_naive_dft(oracle, n, sign):
    x = _rand(n, n)
    assert rel_l2(oracle.fft1d(x, sign), oracle.dft1d(x, sign)) <= 1e-13 or n == 1


@pytest.mark.parametrize("n", [8, 64])
def test_naive_dft_is_the_definition(oracle, n):
    # the definition retyped with exact integer angle reduction in numpy longdouble
    x = _rand(n, 7)
    j = np.arange(n)
    W = np.exp(-2j * np.pi * ((np.outer(j, j) % n) / n))
    assert rel_l2(oracle.dft1d(x, -1), W @ x) <= 1e-13
    assert rel_l2(oracle.dft1d(x, +1), np.conj(W) @ x / n) <= 1e-13


def test_shifted_impulse_pins_the_sign(oracle):
    # x = delta[j-1]  =>  X[k] = exp(-2 pi i k / n) (forward),  exp(+2 pi i k/n)/n (inverse)
    n = 32
    x = np.zeros(n, complex); x[1] = 1
    k = np.arange(n)
    assert np.allclose(oracle.fft1d(x, -1), np.exp(-2j * np.pi * k / n), atol=1e-15)
    assert np.allclose(oracle.fft1d(x, +1), np.exp(+2j * np.pi * k / n) / n, atol=1e-15)


def test_impulse_constant_parseval_roundtrip(oracle):
    n = 256
    d = np.zeros(n, complex); d[0] = 1
    assert np.allclose(oracle.fft1d(d, -1), 1.0, atol=1e-15)
    c = np.ones(n, complex)
    X = oracle.fft1d(c, -1)
    assert abs(X[0] - n) < 1e-12 and np.max(np.abs(X[1:])) < 1e-12
    x = _rand(n, 3)
    X = oracle.fft1d(x, -1)
    assert abs(np.sum(np.abs(X) ** 2) / n / np.sum(np.abs(x) ** 2) - 1) < 1e-14
    assert rel_l2(oracle.fft1d(X, +1), x) <= 1e-14


def test_fft1d_large_vs_numpy_library(oracle):
    # special case that reduces to a library routine (pocketfft), 16384 points
    x = _rand(16384, 11)
    assert rel_l2(oracle.fft1d(x, -1), np.fft.fft(x)) <= 1e-13
    assert rel_l2(oracle.fft1d(x, +1), np.fft.ifft(x)) <= 1e-13


def test_fft1d_rejects_non_power_of_two(oracle):
    with pytest.raises(ValueError):
        oracle.fft1d(np.ones(12, complex))


@pytest.mark.parametrize("shape", [(8, 8), (4, 16), (16, 8)])
@pytest.mark.parametrize("sign", [-1, +1])
def test_fft2d_equals_naive_dft2d(oracle, shape, sign):
    a = _rand(shape, 5)
    assert rel_l2(oracle.fft2d(a, sign), oracle.dft2d(a, sign)) <= 1e-13


def test_fft2d_plane_wave_pins_axes(oracle):
    # a[y][x] = exp(2 pi i (3 x / nx + 5 y / ny))  =>  single bin (l=5, k=3) of height nx*ny.
    ny, nx = 16, 32
    y, x = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    a = np.exp(2j * np.pi * (3 * x / nx + 5 * y / ny))
    A = oracle.fft2d(a, -1)
    ref = np.zeros((ny, nx), complex); ref[5, 3] = nx * ny
    assert np.max(np.abs(A - ref)) < 1e-10
    assert rel_l2(oracle.fft2d(A, +1), a) <= 1e-14


def test_fft2d_threads_do_not_change_bits(oracle):
    a = _rand((64, 128), 9)
    t = oracle.lib().cwo_oracle_get_threads()
    oracle.set_threads(1); r1 = oracle.fft2d(a)
    oracle.set_threads(4); r4 = oracle.fft2d(a)
    oracle.set_threads(t)
    assert np.array_equal(r1, r4)
