"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json configs c1..c5).

This module holds NO arithmetic of the method (no FFT, no transfer function, no propagation):
only random draws and the amplitude/phase -> complex packing that defines an input field.
It serves the oracle (tests) and the CUDA path (tests, bench) alike and imports neither.

The paper's own inputs are 8-bit photographs and a two-dot hologram (P:L246, P:L276,
P:L654-655) that are not available; these generators stand in for them
(recipe: DESIGN.md "Input recipe").  Draws use
numpy.random.Generator(PCG64(seed)), seed = 11075578*10 + config index; amplitude and phase
are formed in double and rounded ONCE to complex64 / float32, and the same arrays go to
the oracle and to the GPU.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import Tuple

import numpy as np

SEED_BASE = 11075578 * 10


@dataclass(frozen=True)
class Config:
    name: str
    op: str                 # "asm" | "fresnel" | "stack" | "gs"
    N: int                  # Nx = Ny
    lam: float              # wavelength [m]
    pitch: float            # sampling pitch [m]
    zs: Tuple[float, ...]   # propagation distance(s) [m]
    iters: int = 0          # GS iterations
    index: int = 0          # seed offset

    def scaled(self, N: int) -> "Config":
        """Same physics on a smaller grid (parity-test sizes)."""
        return replace(self, N=N, name="%s@%d" % (self.name.split("@")[0], N))


CONFIGS = {
    "c1": Config("c1", "asm", 256, 633e-9, 10e-6, (0.05,), index=1),
    "c2": Config("c2", "fresnel", 1024, 532e-9, 8e-6, (0.2,), index=2),
    "c3": Config("c3", "asm", 4096, 633e-9, 4e-6, (0.01, 0.1, 0.5), index=3),
    "c4": Config("c4", "stack", 2048, 633e-9, 6.4e-6, tuple(0.001 * k for k in range(1, 65)), index=4),
    "c5": Config("c5", "gs", 8192, 532e-9, 3.74e-6, (0.3,), iters=20, index=5),
}


def rng_for(cfg: Config, stream: int = 0) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(SEED_BASE + cfg.index + 1000 * stream))


def _pack(amp: np.ndarray, phase: np.ndarray) -> np.ndarray:
    """amplitude, phase (double) -> complex64, rounded once."""
    return (amp * np.exp(1j * phase)).astype(np.complex64)


def field_c1(cfg: Config) -> np.ndarray:
    """a ~ U[0,1), phi ~ U[0,2pi)."""
    r = rng_for(cfg)
    a = r.random((cfg.N, cfg.N))
    ph = r.random((cfg.N, cfg.N)) * (2 * np.pi)
    return _pack(a, ph)


def field_c2(cfg: Config) -> np.ndarray:
    """Binary random-dot aperture, 5% ones (particle-hologram-like)."""
    r = rng_for(cfg)
    return (r.random((cfg.N, cfg.N)) < 0.05).astype(np.complex64)


def field_c3(cfg: Config) -> np.ndarray:
    """Re, Im ~ N(0,1) i.i.d. == Rayleigh(sigma=1) amplitude with uniform phase (speckle)."""
    r = rng_for(cfg)
    out = np.empty((cfg.N, cfg.N), np.complex64)
    out.real = r.standard_normal((cfg.N, cfg.N), dtype=np.float32)
    out.imag = r.standard_normal((cfg.N, cfg.N), dtype=np.float32)
    return out


def field_c4(cfg: Config) -> np.ndarray:
    """|u1| = 1, phi ~ U[0,2pi) (random-phase field)."""
    r = rng_for(cfg)
    ph = r.random((cfg.N, cfg.N)) * (2 * np.pi)
    return _pack(np.ones_like(ph), ph)


def _box_blur_periodic(a: np.ndarray, k: int) -> np.ndarray:
    """k x k periodic box mean (k odd), separable sums of shifted copies."""
    h = k // 2
    acc = np.zeros_like(a)
    for s in range(-h, h + 1):
        acc += np.roll(a, s, axis=0)
    out = np.zeros_like(a)
    for s in range(-h, h + 1):
        out += np.roll(acc, s, axis=1)
    return out / float(k * k)


def gs_inputs_c5(cfg: Config):
    """amp_src == 1; amp_dst = 9x9 periodic box blur of U[0,1) noise scaled to the same energy;
    phi0 ~ U[0,2pi).  Returns float32 arrays (amp_src, amp_dst, phi0)."""
    r = rng_for(cfg)
    n = cfg.N
    amp_src = np.ones((n, n), np.float32)
    noise = r.random((n, n))
    amp_dst = _box_blur_periodic(noise, 9)
    amp_dst *= np.sqrt(float(n) * n / np.sum(amp_dst * amp_dst))
    phi0 = (r.random((n, n)) * (2 * np.pi)).astype(np.float32)
    return amp_src, amp_dst.astype(np.float32), phi0


def gs_inputs(shape, seed: int):
    """gs_inputs_c5's recipe on an arbitrary (Ny, Nx) grid (non-square parity cases): amp_src == 1, amp_dst = 9x9
    periodic box blur of U[0,1) noise scaled to the same energy, phi0 ~ U[0,2pi).  float32 arrays."""
    r = np.random.Generator(np.random.PCG64(SEED_BASE + 5 + 1000 * int(seed)))
    ny, nx = shape
    amp_src = np.ones((ny, nx), np.float32)
    amp_dst = _box_blur_periodic(r.random((ny, nx)), 9)
    amp_dst *= np.sqrt(float(ny) * nx / np.sum(amp_dst * amp_dst))
    phi0 = (r.random((ny, nx)) * (2 * np.pi)).astype(np.float32)
    return amp_src, amp_dst.astype(np.float32), phi0


def random_phasor(cfg: Config, stream: int = 1) -> np.ndarray:
    """Unit-modulus complex64 field with uniform phase (restart states for GS parity)."""
    r = rng_for(cfg, stream)
    ph = r.random((cfg.N, cfg.N)) * (2 * np.pi)
    return _pack(np.ones_like(ph), ph)


FIELD_GENERATORS = {"c1": field_c1, "c2": field_c2, "c3": field_c3, "c4": field_c4}


def make_field(cfg: Config) -> np.ndarray:
    return FIELD_GENERATORS[cfg.name.split("@")[0]](cfg)
