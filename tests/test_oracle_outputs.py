"""Pins for the oracle's output conversions: Scale (Eq.(21)) and the point-light-source CGH
(Eq.(23))."""
import numpy as np

import closed_forms as cf

LAM = 633e-9


def test_scale255_range_and_affine_invariance(oracle):
    r = np.random.default_rng(1)
    a = r.standard_normal((17, 33)) ** 2
    s = oracle.scale255(a)
    assert s.min() == 0.0 and s.max() == 255.0
    assert s.flat[np.argmin(a)] == 0.0 and s.flat[np.argmax(a)] == 255.0
    # Eq.(21) is invariant under I -> alpha I + beta (alpha > 0) and keeps ratios of differences
    assert np.allclose(oracle.scale255(3.5 * a + 11.0), s, rtol=0, atol=1e-10)
    i, j, k = 5, 100, 300
    assert np.isclose((s.flat[i] - s.flat[j]) / (s.flat[k] - s.flat[j]), (a.flat[i] - a.flat[j]) / (a.flat[k] - a.flat[j]))
    assert np.all(oracle.scale255(np.full((4, 4), 2.5)) == 0.0)       # reading R18


def test_pls_single_point_is_a_zone_plate(oracle):
    # one on-axis source: I = A cos(pi r^2/(lambda z)); values against 50-digit arithmetic, incl. Nx != Ny, px != py
    ny, nx, px, py, zj = 48, 64, 4e-6, 3e-6, 0.2
    I = oracle.pls_cgh(ny, nx, px, py, LAM, [0.0], [0.0], [zj], [1.7])
    for (i, j) in [(32, 24), (0, 0), (63, 47), (10, 40), (33, 24), (32, 25)]:
        ref = 1.7 * cf.pls_term(repr(LAM), repr(zj), repr((i - nx // 2) * px), repr((j - ny // 2) * py))
        assert abs(I[j, i] - ref) < 1e-9, (i, j)
    assert I[24, 32] == 1.7                                         # r = 0
    # even in x and y about the centre sample
    assert np.allclose(I[24 + 5, 32 + 7], I[24 - 5, 32 - 7], atol=1e-12)


def test_pls_lateral_shift_sign_and_axes(oracle):
    # a source at (+3 px, -5 py) gives the on-axis pattern translated by (+3, -5) samples
    ny, nx, px, py, zj = 64, 64, 4e-6, 3e-6, 0.05
    a = oracle.pls_cgh(ny, nx, px, py, LAM, [0.0], [0.0], [zj], [1.0])
    b = oracle.pls_cgh(ny, nx, px, py, LAM, [3 * px], [-5 * py], [zj], [1.0])
    assert np.allclose(b[10:40, 10:40], a[15:45, 7:37], atol=1e-9)


def test_pls_superposition_and_depth(oracle):
    ny, nx, p = 32, 32, 4e-6
    xs, ys, zs, am = [10e-6, -33e-6, 0.0], [5e-6, 12e-6, -40e-6], [0.1, 0.15, 0.22], [1.0, 0.5, 2.0]
    tot = oracle.pls_cgh(ny, nx, p, p, LAM, xs, ys, zs, am)
    parts = sum(oracle.pls_cgh(ny, nx, p, p, LAM, [x], [y], [z], [a]) for x, y, z, a in zip(xs, ys, zs, am))
    assert np.allclose(tot, parts, atol=1e-12)
    # the depth enters as 1/z_j: halving z_j doubles the phase => same pattern as doubling both lateral distances^2
    one = oracle.pls_cgh(ny, nx, p, p, LAM, [0.0], [0.0], [0.1], [1.0])
    ref = cf.pls_term(repr(LAM), "0.1", repr(7 * p), repr(-3 * p))
    assert abs(one[16 - 3, 16 + 7] - ref) < 1e-9


def test_intensity_is_re2_plus_im2(oracle):
    # Eq.(20): exact small integers (3-4-5, 5-12-13), unit phasors, |c u|^2 = |c|^2 |u|^2, Parseval against the oracle's own
    # FFT, and the C oracle's stack intensity of one plane (written independently in cwo_oracle.c)
    u = np.array([[3 + 4j, -5 + 12j], [0j, -1j]])
    assert np.array_equal(oracle.intensity(u), np.array([[25.0, 169.0], [0.0, 1.0]]))
    r = np.random.default_rng(3)
    th = r.uniform(0, 2 * np.pi, (8, 16))
    assert np.allclose(oracle.intensity(np.exp(1j * th)), 1.0, rtol=0, atol=1e-15)
    v = r.standard_normal((8, 16)) + 1j * r.standard_normal((8, 16))
    assert np.allclose(oracle.intensity((2 - 1j) * v), 5.0 * oracle.intensity(v), rtol=1e-14)
    assert np.isclose(oracle.intensity(oracle.fft2d(v)).sum(), v.size * oracle.intensity(v).sum(), rtol=1e-13)
    px, lam, z = 4e-6, LAM, 0.003
    assert np.allclose(oracle.intensity(oracle.asm(v, px, px, lam, z)), oracle.stack_intensity(v, px, px, lam, [z])[0],
                       rtol=1e-13, atol=0)


def test_real_field_conversions_of_section_5(oracle):
    # exact cases (3-4-5 triangle, the axes), and the paper's own round trips: Complex(a, b) of conversion 5 rebuilds u from
    # amplitude and phase, conversion 6 from the real and imaginary parts
    u = np.array([[3 + 4j, -3 + 4j, -3 - 4j], [1 + 0j, 1j, -1 + 0j], [-1j, 0j, 2 - 2j]])
    assert np.array_equal(oracle.amplitude(u)[0], [5.0, 5.0, 5.0])
    assert np.array_equal(oracle.re(u)[0], [3.0, -3.0, -3.0]) and np.array_equal(oracle.im(u)[0], [4.0, 4.0, -4.0])
    th = oracle.phase(u)
    assert np.allclose(th[1], [0.0, np.pi / 2, np.pi], atol=1e-15) and np.isclose(th[2, 0], -np.pi / 2)
    assert th[2, 1] == 0.0 and np.isclose(th[2, 2], -np.pi / 4)
    assert np.isclose(th[0, 0], np.arctan(4.0 / 3.0)) and np.isclose(th[0, 1], np.pi - np.arctan(4.0 / 3.0))   # quadrants
    assert np.isclose(th[0, 2], -np.pi + np.arctan(4.0 / 3.0))
    r = np.random.default_rng(5)
    v = r.standard_normal((16, 8)) + 1j * r.standard_normal((16, 8))
    assert np.allclose(oracle.amplitude(v) ** 2, oracle.intensity(v), rtol=1e-14)
    assert np.allclose(oracle.amplitude(v) * np.exp(1j * oracle.phase(v)), v, rtol=1e-13)
    assert np.array_equal(oracle.re(v) + 1j * oracle.im(v), v)
    assert oracle.phase(v).min() >= -np.pi and oracle.phase(v).max() <= np.pi
