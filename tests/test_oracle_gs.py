"""Pins for the oracle's Gerchberg-Saxton loop (Listing 8; SURVEY 8(c) O-GS)."""
import numpy as np
import pytest

from conftest import rel_l2

PX, LAM = 8e-6, 532e-9


def _inputs(n, seed):
    r = np.random.default_rng(seed)
    amp_src = np.ones((n, n))
    amp_dst = r.random((n, n)) + 0.1
    amp_dst *= np.sqrt(n * n / np.sum(amp_dst ** 2))
    phi0 = r.random((n, n)) * 2 * np.pi
    return amp_src, amp_dst, phi0


def _phasor(u):
    a = np.abs(u)
    return np.where(a == 0, 1.0, u / np.where(a == 0, 1, a))


@pytest.mark.parametrize("method", [0, 1])
def test_zero_iterations_is_the_kinoform(oracle, method):
    # iters = 0 returns the phase of P(-z)[amp_dst exp(i phi0)]: the kinoform of section 7.1
    n, z = 32, 0.004
    amp_src, amp_dst, phi0 = _inputs(n, 1)
    P = (lambda u, zz: oracle.asm(u, PX, PX, LAM, zz)) if method else (lambda u, zz: oracle.fresnel_conv(u, PX, PX, LAM, zz))
    ph = oracle.gs(method, amp_src, amp_dst, phi0, PX, PX, LAM, z, 0)
    ref = P(amp_dst * np.exp(1j * phi0), -z)
    assert np.max(np.abs(np.exp(1j * ph) - _phasor(ref))) < 1e-12
    assert ph.min() > -np.pi - 1e-15 and ph.max() <= np.pi


@pytest.mark.parametrize("method", [0, 1])
def test_loop_equals_step_by_step_restatement(oracle, method):
    # The loop of Listing 8 lines 8-17 written out in the test from the separately pinned propagations.
    n, z, iters = 32, 0.004, 3
    amp_src, amp_dst, phi0 = _inputs(n, 2)
    amp_src = amp_src * (1 + 0.3 * np.random.default_rng(5).random((n, n)))     # non-uniform source amplitude
    P = (lambda u, zz: oracle.asm(u, PX, PX, LAM, zz)) if method else (lambda u, zz: oracle.fresnel_conv(u, PX, PX, LAM, zz))
    p = _phasor(P(amp_dst * np.exp(1j * phi0), -z))
    for _ in range(iters):
        G = P(amp_src * p, +z)
        q = _phasor(G)
        p = _phasor(P(amp_dst * q, -z))
    ph = oracle.gs(method, amp_src, amp_dst, phi0, PX, PX, LAM, z, iters)
    assert np.max(np.abs(np.exp(1j * ph) - p)) < 1e-10
    # the split init/iter entry points follow the same trajectory
    p2 = oracle.gs_init(method, amp_dst, phi0, PX, PX, LAM, z)
    for _ in range(iters):
        p2 = oracle.gs_iter(method, amp_src, amp_dst, p2, PX, PX, LAM, z)
    assert np.max(np.abs(p2 - p)) < 1e-10


def test_error_is_non_increasing_with_unitary_asm(oracle):
    # With the unpadded ASM propagator (unitary) the GS error cannot increase (Fienup, ref [18] P:L808).
    n, z = 64, 0.003
    amp_src, amp_dst, phi0 = _inputs(n, 3)
    p = oracle.gs_init(1, amp_dst, phi0, PX, PX, LAM, z)
    errs = [oracle.gs_error(1, amp_src, amp_dst, p, PX, PX, LAM, z)]
    for _ in range(8):
        p = oracle.gs_iter(1, amp_src, amp_dst, p, PX, PX, LAM, z)
        errs.append(oracle.gs_error(1, amp_src, amp_dst, p, PX, PX, LAM, z))
    assert all(b <= a + 1e-12 for a, b in zip(errs, errs[1:])), errs
    assert errs[-1] < 0.8 * errs[0]
    # gs_error is what it says: recompute from G of one more pass
    p3, G = oracle.gs_iter(1, amp_src, amp_dst, p, PX, PX, LAM, z, want_G=True)
    e = np.linalg.norm(np.abs(G) - amp_dst) / np.linalg.norm(amp_dst)
    assert abs(e - errs[-1]) < 1e-12


def test_consistent_pair_is_a_fixed_point(oracle):
    # If amp_dst = |P(+z)[amp_src p*]| for some phasor p*, then starting from the phase of that
    # reconstruction the loop stays put and the error is 0 (unitary ASM).
    n, z = 32, 0.002
    r = np.random.default_rng(7)
    amp_src = np.ones((n, n))
    pstar = np.exp(2j * np.pi * r.random((n, n)))
    G = oracle.asm(amp_src * pstar, PX, PX, LAM, z)
    amp_dst = np.abs(G)
    phi0 = np.angle(G)
    ph = oracle.gs(1, amp_src, amp_dst, phi0, PX, PX, LAM, z, 4)
    assert np.max(np.abs(np.exp(1j * ph) - pstar)) < 1e-9
    assert oracle.gs_error(1, amp_src, amp_dst, pstar, PX, PX, LAM, z) < 1e-12


def test_zero_sample_has_phase_zero(oracle):
    # phasor(0) = 1 (atan2(0,0) = 0, Eq.(25)): an all-zero target gives phase 0 everywhere
    n = 16
    ph = oracle.gs(1, np.ones((n, n)), np.zeros((n, n)), np.ones((n, n)), PX, PX, LAM, 0.001, 0)
    assert np.all(ph == 0)


def test_fresnel_error_trend(oracle):
    # Fresnel conv is not unitary (aliased impulse response) so monotonicity is not guaranteed, but the
    # paper's claim "gradually improve the quality" holds for the c5-like regime.
    n, px, z = 64, 3.74e-6, 0.3 * (64 / 8192)      # keeps N pitch^2/(lambda z) = 0.718 as in c5
    amp_src, amp_dst, phi0 = _inputs(n, 9)
    p = oracle.gs_init(0, amp_dst, phi0, px, px, LAM, z)
    e0 = oracle.gs_error(0, amp_src, amp_dst, p, px, px, LAM, z)
    for _ in range(10):
        p = oracle.gs_iter(0, amp_src, amp_dst, p, px, px, LAM, z)
    assert oracle.gs_error(0, amp_src, amp_dst, p, px, px, LAM, z) < e0
