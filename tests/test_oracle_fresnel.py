"""Pins for the oracle's convolution-form Fresnel diffraction (Eq.(1)-(6))."""
import numpy as np
import pytest

import closed_forms as cf
from conftest import rel_l2
from test_oracle_asm import _pins


def _rand(shape, seed):
    r = np.random.default_rng(seed)
    return r.standard_normal(shape) + 1j * r.standard_normal(shape)


@pytest.mark.parametrize("pin", _pins("FRES"))
def test_closed_form_delta_matches_survey_pins(pin):
    _, lam, d, z, dm, dn, re, im = pin
    v = cf.fresnel_delta(d, d, lam, z, dm, dn)
    assert abs(v - complex(re, im)) < 1e-15


@pytest.mark.parametrize("pin", _pins("GAUSS"))
def test_closed_form_gaussian_matches_survey_pins(pin):
    _, lam, d, z, m, n, re, im = pin
    dd = float(d)
    v = cf.gaussian_beam(lam, z, "120e-6", repr(m * dd), repr(n * dd))
    assert abs(v - complex(re, im)) < 1e-9


@pytest.mark.parametrize("shape,px,py,z", [((16, 16), 8e-6, 8e-6, 0.002), ((16, 32), 6e-6, 9e-6, -0.003),
                                          ((32, 16), 8e-6, 5e-6, 0.0011)])
def test_fft_pipeline_equals_direct_linear_convolution(oracle, shape, px, py, z):
    # pins pad / wrap / crop / centring of the literal Eq.(5) pipeline
    u1 = _rand(shape, 1)
    a = oracle.fresnel_conv(u1, px, py, 532e-9, z)
    b = oracle.fresnel_direct(u1, px, py, 532e-9, z)
    assert rel_l2(a, b) < 1e-12
    ny, nx = shape
    ms = np.array([0, nx - 1, 3]); ns = np.array([0, ny - 1, 5])
    c = oracle.fresnel_points(u1, px, py, 532e-9, z, ms, ns)
    assert np.allclose(c, b[ns, ms], rtol=0, atol=1e-14 * np.abs(b).max())


def test_delta_response_is_c_times_hF(oracle):
    # u1 = delta at (m0, n0)  =>  u2[n, m] = c * h_F(m - m0, n - n0): pins prefactor, sign, pitch^2,
    # and (with px != py, Nx != Ny) which axis is which.
    ny, nx, px, py, lam, z = 64, 128, 8e-6, 5e-6, 532e-9, 0.02
    m0, n0 = 40, 17
    u1 = np.zeros((ny, nx), complex); u1[n0, m0] = 1
    u2 = oracle.fresnel_conv(u1, px, py, lam, z)
    for (m, n) in [(40, 17), (0, 0), (127, 63), (41, 17), (40, 18), (100, 3)]:
        ref = cf.fresnel_delta(repr(px), repr(py), repr(lam), repr(z), m - m0, n - n0)
        assert abs(u2[n, m] - ref) < 1e-10 * abs(ref), (m, n)   # z/lambda ~ 4e4 cycles in double
    assert abs(abs(u2[0, 0]) - px * py / (lam * z)) < 1e-15


def test_delta_response_c2_survey_value(oracle):
    # c2 parameters, offset (100, -37) => (5.97279959666158e-4, 7.11577286857595e-5)
    N = 256
    u1 = np.zeros((N, N), complex); u1[100, 50] = 1
    v = oracle.fresnel_points(u1, 8e-6, 8e-6, 532e-9, 0.2, [150], [63])[0]
    assert abs(v - complex(5.97279959666158e-4, 7.11577286857595e-5)) < 1e-11
    # back-propagation pin (z = -0.3, c5 pitch)
    v = oracle.fresnel_points(u1, 3.74e-6, 3.74e-6, 532e-9, -0.3, [150], [63])[0]
    assert abs(v - complex(8.67567720556418e-5, -1.24222886754195e-5)) < 1e-11


def test_gaussian_beam_closed_form(oracle):
    # u1 = exp(-r^2/w0^2) => u2 = exp(ikz) (1/q) exp(-r^2/(w0^2 q)), q = 1 + i z/z_R (S8c Fresnel pin iii)
    N, d, lam, z, w0 = 256, 8e-6, 532e-9, 0.05, 120e-6
    c = (np.arange(N) - N // 2) * d
    u1 = np.exp(-(c[None, :] ** 2 + c[:, None] ** 2) / w0 ** 2)
    u2 = oracle.fresnel_conv(u1, d, d, lam, z)
    zR = np.pi * w0 ** 2 / lam
    q = 1 + 1j * z / zR
    kz = z / lam
    ref = np.exp(2j * np.pi * (kz - np.floor(kz))) / q * np.exp(-(c[None, :] ** 2 + c[:, None] ** 2) / (w0 ** 2 * q))
    assert rel_l2(u2, ref) < 1e-11
    # two samples in 50-digit arithmetic
    for (m, n) in [(0, 0), (10, -7)]:
        v = cf.gaussian_beam("532e-9", "0.05", "120e-6", repr(m * d), repr(n * d))
        assert abs(u2[N // 2 + n, N // 2 + m] - v) < 1e-10
    # ~unitary: energy conserved because pitch^2 is included (reading R6)
    assert abs(np.sum(np.abs(u2) ** 2) / np.sum(np.abs(u1) ** 2) - 1) < 1e-10


def test_adjoint_identity_pins_minus_z(oracle):
    # <P(z) a, b> = <a, P(-z) b>: back-propagation is the adjoint (S8c Fresnel pin v)
    a = _rand((32, 32), 2); b = _rand((32, 32), 3)
    px, lam, z = 8e-6, 532e-9, 0.004
    lhs = np.vdot(b, oracle.fresnel_conv(a, px, px, lam, z))          # sum conj(b) * P(z)a
    rhs = np.vdot(oracle.fresnel_conv(b, px, px, lam, -z), a)         # sum conj(P(-z)b) * a
    assert abs(lhs - rhs) < 1e-13 * abs(lhs)


def test_convolution_theorem_rank1_spectrum(oracle):
    # FFT2 of the sampled 2-D h_F == outer product of the 1-D chirp FFTs (S8c Fresnel pin vi)
    N, d, lam, z = 16, 8e-6, 532e-9, 0.001
    taps = np.where(np.arange(2 * N) < N, np.arange(2 * N), np.arange(2 * N) - 2 * N)
    h1 = np.exp(1j * np.pi * (taps * d) ** 2 / (lam * z))
    H2 = oracle.fft2d(np.outer(h1, h1))
    C = oracle.fft1d(h1)
    assert rel_l2(H2, np.outer(C, C)) < 1e-13


def test_linearity_and_shift_invariance(oracle):
    a = _rand((16, 16), 5); b = _rand((16, 16), 6)
    P = lambda u: oracle.fresnel_conv(u, 8e-6, 8e-6, 532e-9, 0.002)
    assert rel_l2(P(2 * a - 3j * b), 2 * P(a) - 3j * P(b)) < 1e-13


def test_z_zero_is_an_error(oracle):
    with pytest.raises(ValueError):
        oracle.fresnel_conv(np.ones((16, 16), complex), 8e-6, 8e-6, 532e-9, 0.0)
