"""Pins for the oracle's Fresnel diffraction between planes of different pitch / offset: the direct sum of Eq.(1),
the Fourier form (Eq.(7)-(9)) and the shifted Fresnel diffraction (Eq.(10)-(14))."""
import numpy as np
import pytest

import closed_forms as cf
from conftest import rel_l2

LAM = 532e-9


def _rand(shape, seed):
    r = np.random.default_rng(seed)
    return r.standard_normal(shape) + 1j * r.standard_normal(shape)


def test_general_direct_reduces_to_the_convolution_form(oracle):
    # equal pitches, no offset: the sum IS Eq.(1) on one grid = the (pinned) direct linear convolution
    u1 = _rand((16, 32), 3)
    a = oracle.fresnel_general_direct(u1, (8e-6, 5e-6), (8e-6, 5e-6), LAM, 0.004)
    b = oracle.fresnel_direct(u1, 8e-6, 5e-6, LAM, 0.004)
    assert rel_l2(a, b) < 1e-12


@pytest.mark.parametrize("z", [0.03, -0.021])
def test_general_delta_response_closed_form(oracle, z):
    # one source sample at index (m0, n0): u2 = c exp(i pi ((x1-x0)^2 + (y1-y0)^2)/(lambda z)) with
    # x0 = (m0 - Nx/2) p0x + O0x, x1 = (m1 - Nx/2) p1x + O1x: pins pitches, both offsets and their signs,
    # the centring of Eq.(4), which axis is which (Nx != Ny, px != py), the prefactor and the area element
    ny, nx = 32, 64
    p0, p1, o0, o1 = (8e-6, 5e-6), (3e-6, 11e-6), (20e-6, -35e-6), (-140e-6, 75e-6)
    m0, n0 = 40, 9
    u1 = np.zeros((ny, nx), complex); u1[n0, m0] = 1
    u2 = oracle.fresnel_general_direct(u1, p0, p1, LAM, z, o0, o1)
    x0 = (m0 - nx // 2) * p0[0] + o0[0]; y0 = (n0 - ny // 2) * p0[1] + o0[1]
    for (m1, n1) in [(0, 0), (63, 31), (32, 16), (5, 30), (41, 9)]:
        x1 = (m1 - nx // 2) * p1[0] + o1[0]; y1 = (n1 - ny // 2) * p1[1] + o1[1]
        ref = cf.fresnel_delta_xy(repr(p0[0]), repr(p0[1]), repr(LAM), repr(z), repr(x1 - x0), repr(y1 - y0))
        assert abs(u2[n1, m1] - ref) < 1e-9 * abs(ref), (m1, n1)
    pts = oracle.fresnel_general_points(u1, p0, p1, LAM, z, [0, 63, 5], [0, 31, 30], o0, o1)
    assert np.allclose(pts, u2[[0, 31, 30], [0, 63, 5]], rtol=0, atol=1e-14 * np.abs(u2).max())


def test_general_points_gaussian_beam_closed_form(oracle):
    # Gaussian exp(-r^2/w0^2) centred on the optical axis, sampled on an OFFSET source grid, observed on a grid of
    # another pitch and offset: the Fresnel integral has the closed form exp(ikz)/q exp(-r^2/(w0^2 q))
    n, p0, p1, z, w0 = 256, (8e-6, 8e-6), (5e-6, 6e-6), 0.05, 120e-6
    o0, o1 = (24e-6, -16e-6), (37e-6, -52e-6)
    j = np.arange(n) - n // 2
    x0 = j * p0[0] + o0[0]; y0 = j * p0[1] + o0[1]
    u1 = np.exp(-(x0[None, :] ** 2 + y0[:, None] ** 2) / w0 ** 2)
    ms = np.array([128, 100, 160, 128, 90]); ns = np.array([128, 128, 120, 150, 170])
    got = oracle.fresnel_general_points(u1, p0, p1, LAM, z, ms, ns, o0, o1)
    for g, m, k in zip(got, ms, ns):
        x1 = (m - n // 2) * p1[0] + o1[0]; y1 = (k - n // 2) * p1[1] + o1[1]
        ref = cf.gaussian_beam(repr(LAM), repr(z), repr(w0), repr(float(x1)), repr(float(y1)))
        assert abs(g - ref) < 1e-9, (m, k)


@pytest.mark.parametrize("z", [0.02, -0.015])
def test_shifted_algorithm_equals_the_direct_sum(oracle, z):
    # Eq.(10)-(14) step by step against the sum it evaluates: pins every chirp / ramp factor of Eq.(11)-(13),
    # the units of the offsets (reading R16) and the linear (2N-expanded) convolution
    u1 = _rand((16, 32), 5)
    p0, p1, o0, o1 = (8e-6, 5e-6), (3e-6, 7e-6), (12e-6, -9e-6), (-60e-6, 44e-6)
    a = oracle.fresnel_shifted(u1, p0, p1, LAM, z, o0, o1)
    b = oracle.fresnel_general_direct(u1, p0, p1, LAM, z, o0, o1)
    assert rel_l2(a, b) < 1e-11


def test_shifted_with_equal_pitch_and_no_offset_is_the_convolution_form(oracle):
    u1 = _rand((64, 64), 6)
    a = oracle.fresnel_shifted(u1, (8e-6, 6e-6), (8e-6, 6e-6), LAM, 0.01)
    b = oracle.fresnel_conv(u1, 8e-6, 6e-6, LAM, 0.01)
    assert rel_l2(a, b) < 1e-11


@pytest.mark.parametrize("z", [0.004, -0.0031])
def test_fourier_form_equals_the_direct_sum_at_its_destination_pitch(oracle, z):
    # destination pitch lambda |z| / (N p) (reading R17); z < 0 turns the transform into the inverse kernel
    ny, nx, px, py = 16, 32, 8e-6, 5e-6
    u1 = _rand((ny, nx), 7)
    a = oracle.fresnel_fourier(u1, px, py, LAM, z)
    p1 = (LAM * abs(z) / (nx * px), LAM * abs(z) / (ny * py))
    b = oracle.fresnel_general_direct(u1, (px, py), p1, LAM, z)
    assert rel_l2(a, b) < 1e-11


def test_fourier_form_equals_shifted_fresnel_at_that_pitch(oracle):
    n, p, z = 128, 8e-6, 0.03
    u1 = _rand((n, n), 8)
    p1 = LAM * z / (n * p)
    a = oracle.fresnel_fourier(u1, p, p, LAM, z)
    b = oracle.fresnel_shifted(u1, (p, p), (p1, p1), LAM, z)
    assert rel_l2(a, b) < 1e-10


def test_fourier_form_gaussian_beam_closed_form(oracle):
    n, p, z, w0 = 256, 8e-6, 0.05, 120e-6
    j = np.arange(n) - n // 2
    u1 = np.exp(-((j * p)[None, :] ** 2 + (j * p)[:, None] ** 2) / w0 ** 2)
    u2 = oracle.fresnel_fourier(u1, p, p, LAM, z)
    p2 = LAM * z / (n * p)
    for (m, k) in [(128, 128), (120, 128), (128, 140), (110, 150)]:
        ref = cf.gaussian_beam(repr(LAM), repr(z), repr(w0), repr((m - n // 2) * p2), repr((k - n // 2) * p2))
        assert abs(u2[k, m] - ref) < 1e-9, (m, k)


def test_fourier_form_delta_response(oracle):
    ny, nx, px, py, z = 32, 64, 8e-6, 5e-6, 0.01
    m0, n0 = 21, 30
    u1 = np.zeros((ny, nx), complex); u1[n0, m0] = 1
    u2 = oracle.fresnel_fourier(u1, px, py, LAM, z)
    p2x, p2y = LAM * z / (nx * px), LAM * z / (ny * py)
    for (m1, n1) in [(0, 0), (63, 31), (40, 3)]:
        dx = (m1 - nx // 2) * p2x - (m0 - nx // 2) * px; dy = (n1 - ny // 2) * p2y - (n0 - ny // 2) * py
        ref = cf.fresnel_delta_xy(repr(px), repr(py), repr(LAM), repr(z), repr(dx), repr(dy))
        assert abs(u2[n1, m1] - ref) < 1e-9 * abs(ref), (m1, n1)
