"""Pins for the oracle's angular spectrum method (Eq.(15)-(17))."""
import os

import numpy as np
import pytest

import closed_forms as cf
from conftest import rel_l2

GOLD = os.path.join(os.path.dirname(__file__), "golden", "survey_pins.txt")


def _pins(kind):
    rows = []
    for line in open(GOLD):
        if line.startswith("#") or not line.strip():
            continue
        t = line.split()
        if t[0] == kind:
            rows.append((int(t[1]), t[2], t[3], t[4], int(t[5]), int(t[6]), float(t[7]), float(t[8])))
    return rows


def _rand(shape, seed):
    r = np.random.default_rng(seed)
    return (r.standard_normal(shape) + 1j * r.standard_normal(shape)).astype(np.complex64)


@pytest.mark.parametrize("pin", _pins("ASM"))
def test_closed_form_module_matches_survey_pins(pin):
    N, lam, d, z, k, l, re, im = pin
    H = cf.asm_H(N, N, d, d, lam, z, k, l)
    assert abs(H - complex(re, im)) < 1e-12


@pytest.mark.parametrize("pin", _pins("ASM"))
def test_transfer_function_entries_match_50_digit_values(oracle, pin):
    N, lam, d, z, k, l, re, im = pin
    H = oracle.asm_transfer(N, N, float(d), float(d), float(lam), float(z))
    # FFT-order storage: negative bins wrap to the top
    assert abs(H[l % N, k % N] - complex(re, im)) < 2e-8      # inputs rounded to double: <~1e-9 moves


def test_plane_wave_is_an_eigenfunction_with_eigenvalue_H(oracle):
    # u1 = exp(i 2 pi (k0 jx / Nx + l0 jy / Ny))  =>  u2 = H(k0, l0) u1 exactly.
    # Nx != Ny, px != py and k0 != l0, negative l0: pins axis wiring, bin->frequency map and sign.
    ny, nx, px, py, lam, z = 32, 64, 3e-6, 5e-6, 633e-9, 0.0123
    jy, jx = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    for (k0, l0) in [(3, -5), (-17, 9), (0, 0), (-32, -16), (31, 15)]:
        u1 = np.exp(2j * np.pi * (k0 * jx / nx + l0 * jy / ny))
        u2 = oracle.asm(u1, px, py, lam, z)
        H = cf.asm_H(nx, ny, repr(px), repr(py), repr(lam), repr(z), k0, l0)
        assert np.max(np.abs(u2 - H * u1)) < 1e-9, (k0, l0)


def test_z0_identity_parseval_roundtrip_semigroup(oracle):
    u1 = _rand((64, 128), 1).astype(np.complex128)
    px, py, lam = 4e-6, 4e-6, 633e-9
    assert rel_l2(oracle.asm(u1, px, py, lam, 0.0), u1) < 1e-15
    u2 = oracle.asm(u1, px, py, lam, 0.01)
    assert abs(np.linalg.norm(u2) / np.linalg.norm(u1) - 1) < 1e-13       # no evanescent bin here
    assert rel_l2(oracle.asm(u2, px, py, lam, -0.01), u1) < 1e-12
    a = oracle.asm(oracle.asm(u1, px, py, lam, 0.004), px, py, lam, 0.006)
    assert rel_l2(a, u2) < 1e-11


@pytest.mark.parametrize("shape", [(8, 8), (8, 16)])
def test_naive_dft_brute_force(oracle, shape):
    u1 = _rand(shape, 2)
    a = oracle.asm(u1, 2e-6, 3e-6, 633e-9, 1e-4)
    b = oracle.asm(u1, 2e-6, 3e-6, 633e-9, 1e-4, naive=True)
    assert rel_l2(a, b) < 1e-12
    # and the definition once more in numpy, with the test's own H from mpmath
    ny, nx = shape
    H = np.array([[cf.asm_H(nx, ny, "2e-6", "3e-6", "633e-9", "1e-4",
                            k if k < nx // 2 else k - nx, l if l < ny // 2 else l - ny)
                   for k in range(nx)] for l in range(ny)])
    c = np.fft.ifft2(np.fft.fft2(u1.astype(complex)) * H)
    assert rel_l2(a, c) < 1e-12


def test_evanescent_components_are_zeroed(oracle):
    # pitch 0.3 um < lambda/sqrt(2): bins with f > 1/lambda exist.  (S8c A2/A4 test config)
    n, d, lam, z = 64, 0.3e-6, 633e-9, 5e-6
    df = 1.0 / (n * d)
    H = oracle.asm_transfer(n, n, d, d, lam, z)
    k = np.fft.fftfreq(n, 1.0 / n)
    w = 1 / lam ** 2 - ((k[None, :] * df) ** 2 + (k[:, None] * df) ** 2)
    assert np.all(H[w < 0] == 0) and np.all(np.abs(np.abs(H[w >= 0]) - 1) < 1e-14)
    assert (w < 0).sum() > 100 and (w >= 0).sum() > 100
    jy, jx = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
    k0, l0 = 25, 20                       # f0 = 32.0 * df = 1.67e6 > 1/lambda = 1.58e6
    assert 1 / lam ** 2 - (k0 ** 2 + l0 ** 2) * df ** 2 < 0
    u1 = np.exp(2j * np.pi * (k0 * jx + l0 * jy) / n)
    assert np.max(np.abs(oracle.asm(u1, d, d, lam, z))) < 1e-12
    k0, l0 = 20, -10                      # inside the circle: still an eigenfunction
    u1 = np.exp(2j * np.pi * (k0 * jx + l0 * jy) / n)
    Hc = cf.asm_H(n, n, "0.3e-6", "0.3e-6", "633e-9", "5e-6", k0, l0)
    assert np.max(np.abs(oracle.asm(u1, d, d, lam, z) - Hc * u1)) < 1e-10
    # back-propagation must not blow up either (z < 0)
    assert np.max(np.abs(oracle.asm_transfer(n, n, d, d, lam, -z))) <= 1 + 1e-14


def test_rayleigh_sommerfeld_sanity(oracle):
    # ASM "calculates the exact solution in scalar light propagation": compare with the
    # RS-I quadrature on a Gaussian well inside the window.  ASM is periodic, RS is not: sanity only.
    # pitch < lambda/2 so the sampled RS kernel is alias-free; then the two agree to ~1e-6.
    n, d, lam, z, w0 = 64, 0.25e-6, 633e-9, 10e-6, 2e-6
    c = (np.arange(n) - n // 2) * d
    u1 = np.exp(-(c[None, :] ** 2 + c[:, None] ** 2) / w0 ** 2)
    a = oracle.asm(u1, d, d, lam, z)
    b = oracle.rs_direct(u1, d, d, lam, z)
    assert rel_l2(a, b) < 1e-4


def test_stack_is_independent_asm_calls(oracle):
    u1 = _rand((32, 32), 4)
    zs = [0.001, 0.002, -0.0015]
    s = oracle.stack(u1, 6.4e-6, 6.4e-6, 633e-9, zs)
    for i, z in enumerate(zs):
        assert np.array_equal(s[i], oracle.asm(u1, 6.4e-6, 6.4e-6, 633e-9, z))
    # semigroup across planes: plane(z1+z2) = asm(plane(z1), z2)
    assert rel_l2(oracle.asm(s[0], 6.4e-6, 6.4e-6, 633e-9, 0.001), s[1]) < 1e-11
