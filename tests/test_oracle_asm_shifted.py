"""Pins of the oracle's shifted / band-limited angular spectrum method (Eq.(18)-(19))
and of the intensity stack (Eq.(20)).  None of them re-types the oracle's own criterion: the band edge
comes from the closed form of the paper's Ref.[56], the rest are reductions to the pinned asm and invariants."""
import numpy as np
import pytest


def _rand(shape, seed):
    r = np.random.default_rng(seed)
    return (r.standard_normal(shape) + 1j * r.standard_normal(shape)).astype(np.complex64)


def _plane_wave(ny, nx, k0, l0):
    jy, jx = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    return np.exp(2j * np.pi * (k0 * jx / nx + l0 * jy / ny))


def test_short_distance_on_axis_is_the_plain_method(oracle):
    # 2 df z << 1: the band 1/(lambda sqrt((2 df z)^2 + 1)) exceeds the Nyquist frequency, nothing is cut
    u1 = _rand((32, 64), 1)
    px, py, lam, z = 4e-6, 5e-6, 633e-9, 1e-4
    assert np.allclose(oracle.asm_shifted(u1, px, py, lam, z), oracle.asm(u1, px, py, lam, z), rtol=0, atol=1e-12)


@pytest.mark.parametrize("z", [3.5e-3, -3.5e-3])
def test_band_edge_is_the_closed_form_of_ref56(oracle, z):
    # on axis the limit is f_lim = 1 / (lambda sqrt((2 df z)^2 + 1)) (band-limited angular spectrum method): a plane
    # wave in bin k is an eigenfunction with eigenvalue H for |k df| <= f_lim and is removed entirely beyond it
    n, p, lam = 64, 4e-6, 633e-9
    df = 1.0 / (n * p)
    f_lim = 1.0 / (lam * np.sqrt((2 * df * z) ** 2 + 1))
    k_lim = int(np.floor(f_lim / df))
    assert 2 < k_lim < n // 2 - 2                    # the edge is inside the grid for these parameters
    for k0, inside in ((k_lim, True), (-k_lim, True), (k_lim + 1, False), (-k_lim - 1, False)):
        for axis in (0, 1):
            kk, ll = (k0, 2) if axis == 0 else (2, k0)
            u1 = _plane_wave(n, n, kk, ll)
            u2 = oracle.asm_shifted(u1, p, p, lam, z)
            if inside:
                w = 1 / lam ** 2 - (kk * df) ** 2 - (ll * df) ** 2
                ph = z * np.sqrt(w)
                H = np.exp(2j * np.pi * (ph - np.floor(ph)))
                assert np.allclose(u2, H * u1, rtol=0, atol=1e-10)
            else:
                assert np.max(np.abs(u2)) < 1e-12


def test_offset_by_whole_pitches_is_a_circular_shift(oracle):
    # exp(i 2 pi O f) in the spectrum samples the propagated field at x + O (sign of the ramp of Eq.(19))
    u1 = _rand((32, 32), 3)
    p, lam, z = 6e-6, 532e-9, 2e-4
    ref = oracle.asm(u1, p, p, lam, z)
    got = oracle.asm_shifted(u1, p, p, lam, z, ox=3 * p, oy=-2 * p)
    assert np.allclose(got, np.roll(np.roll(ref, -3, axis=1), 2, axis=0), rtol=0, atol=1e-11)


def test_offset_moves_the_band_and_z_mirrors_it(oracle):
    n, p, lam, z = 64, 4e-6, 633e-9, 3.5e-3
    df = 1.0 / (n * p)
    S = 0.5 / df
    ox = 0.6 * S                                      # band: |ox - z f / sqrt(1/lam^2 - f^2)| <= S, i.e. f(t), t in [ox - S, ox + S]
    f = lambda t: t / (lam * np.sqrt(t * t + z * z))  # noqa: E731  (Ref.[56]'s u_limit as a function of the edge)
    lo, hi = int(np.ceil(f(ox - S) / df)), int(np.floor(f(ox + S) / df))
    assert lo < 0 < hi and -lo != hi
    keep = lambda k0, zz: np.max(np.abs(oracle.asm_shifted(_plane_wave(n, n, k0, 0), p, p, lam, zz, ox=ox))) > 0.5  # noqa: E731
    assert keep(hi, z) and not keep(hi + 1, z) and keep(lo, z) and not keep(lo - 1, z)
    # back-propagation mirrors the band: g changes sign with z
    assert keep(-hi, -z) and not keep(-hi - 1, -z) and keep(-lo, -z) and not keep(-lo + 1, -z)


def test_mask_only_removes_energy(oracle):
    u1 = _rand((64, 64), 5)
    p, lam = 4e-6, 633e-9
    e0 = np.linalg.norm(u1.astype(np.complex128))
    prev = e0
    for z in (2e-3, 5e-3, 2e-2):
        e = np.linalg.norm(oracle.asm_shifted(u1, p, p, lam, z))
        assert e <= prev * (1 + 1e-12)
        prev = e
    assert prev < 0.9 * e0


def test_intensity_stack(oracle):
    u1 = _rand((32, 64), 7)
    px, py, lam = 6.4e-6, 5e-6, 633e-9
    zs = [0.001, -0.002, 0.03]
    I = oracle.stack_intensity(u1, px, py, lam, zs)
    ref = oracle.stack(u1, px, py, lam, zs)
    assert I.dtype == np.float64 and np.array_equal(I, ref.real ** 2 + ref.imag ** 2)
    assert np.allclose(I.sum(axis=(1, 2)), np.sum(np.abs(u1.astype(np.complex128)) ** 2), rtol=1e-12)   # Parseval
