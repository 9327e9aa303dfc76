"""Pins for the oracle's zero-expanded angular spectrum method (Table 2).

Independent of the oracle's pipeline: H comes from the 50-digit closed form (closed_forms.py), the
impulse response from numpy's FFT of that H, the linear convolution from a direct double sum."""
import numpy as np
import pytest

import closed_forms as cf
from conftest import rel_l2


def _rand(shape, seed):
    r = np.random.default_rng(seed)
    return r.standard_normal(shape) + 1j * r.standard_normal(shape)


def _impulse_response(ny, nx, px, py, lam, z):
    """h on the 2Ny x 2Nx grid: inverse DFT (numpy) of the closed-form H sampled at 1/(2 N p)."""
    my, mx = 2 * ny, 2 * nx
    H = np.empty((my, mx), np.complex128)
    for l in range(my):
        ls = l if l < my // 2 else l - my
        for k in range(mx):
            ks = k if k < mx // 2 else k - mx
            H[l, k] = cf.asm_H(mx, my, px, py, lam, z, ks, ls)
    return np.fft.ifft2(H)


PARAMS = [(8, 8, 10e-6, 10e-6, 633e-9, 0.002), (4, 16, 6e-6, 9e-6, 532e-9, -0.001), (16, 8, 0.4e-6, 0.4e-6, 633e-9, 3e-6)]


@pytest.mark.parametrize("ny,nx,px,py,lam,z", PARAMS)
def test_delta_response_is_the_2n_impulse_response(oracle, ny, nx, px, py, lam, z):
    """A delta at (m0, n0) comes out as h[(m - m0) mod 2Ny, (n - n0) mod 2Nx]: pins the 1/(2Np) sampling, the
    signs, and that the crop is the window the input sat in."""
    h = _impulse_response(ny, nx, px, py, lam, z)
    for m0, n0 in ((0, 0), (ny - 1, 2), (ny // 2, nx - 1)):
        u1 = np.zeros((ny, nx), np.complex128); u1[m0, n0] = 1.0
        got = oracle.asm_pad2x(u1, px, py, lam, z)
        m = (np.arange(ny)[:, None] - m0) % (2 * ny); n = (np.arange(nx)[None, :] - n0) % (2 * nx)
        assert rel_l2(got, h[m, n]) <= 1e-10       # double phase of ~3e3 cycles: ~1e-12


@pytest.mark.parametrize("ny,nx,px,py,lam,z", PARAMS)
def test_equals_the_direct_aperiodic_convolution(oracle, ny, nx, px, py, lam, z):
    """u2[m,n] = sum u1[m1,n1] h[m-m1, n-n1] over the window, offsets |d| < N taken from the 2N-periodic h: the
    expansion removes every wrapped term (what P:L235 introduces it for)."""
    h = _impulse_response(ny, nx, px, py, lam, z)
    u1 = _rand((ny, nx), 5)
    ref = np.zeros((ny, nx), np.complex128)
    for m in range(ny):
        for n in range(nx):
            acc = 0j
            for m1 in range(ny):
                for n1 in range(nx):
                    acc += u1[m1, n1] * h[(m - m1) % (2 * ny), (n - n1) % (2 * nx)]
            ref[m, n] = acc
    assert rel_l2(oracle.asm_pad2x(u1, px, py, lam, z), ref) <= 1e-10


def test_z0_identity_and_energy(oracle):
    u1 = _rand((16, 32), 7)
    assert rel_l2(oracle.asm_pad2x(u1, 5e-6, 7e-6, 633e-9, 0.0), u1) <= 1e-14
    for z in (0.001, 0.05, -0.02):
        u2 = oracle.asm_pad2x(u1, 5e-6, 7e-6, 633e-9, z)
        assert np.linalg.norm(u2) <= np.linalg.norm(u1) * (1 + 1e-12)      # H is unitary on 2N, the crop only loses


def test_differs_from_the_circular_form_by_the_wrapped_terms(oracle):
    """Far enough that light leaves the window: the unpadded call wraps it around, the expanded one does not."""
    n, p, lam, z = 32, 4e-6, 633e-9, 0.002
    u1 = np.zeros((n, n), np.complex128); u1[2:6, 2:6] = 1.0
    a, b = oracle.asm(u1, p, p, lam, z), oracle.asm_pad2x(u1, p, p, lam, z)
    assert rel_l2(a, b) > 1e-2
