"""ctypes face of oracle/cwo_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this module.  It imports nothing from paper_1107_5578_b200 and the package
imports nothing from here.  All arithmetic lives in cwo_oracle.c (double precision);
this file only marshals numpy arrays.

Citations: P:Lnnn = /root/reference/PAPER.md line nnn.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import sys

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "cwo_oracle.c")
_SO = os.path.join(_HERE, "libcwo_oracle.so")

METHOD_FRESNEL = 0   # config c5 (BASELINE.json configs[4])
METHOD_ASM = 1       # the paper's own Listing 8


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp the oracle into oracle/libcwo_oracle.so (rebuilds when the source is newer)."""
    if (not force and os.path.exists(_SO)
            and os.path.getmtime(_SO) >= os.path.getmtime(_SRC)):
        return _SO
    tmp = _SO + ".tmp%d" % os.getpid()
    cmd = ["gcc", "-std=c99", "-O2", "-fopenmp", "-fno-fast-math", "-ffp-contract=off",
           "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, _SO)
    return _SO


_lib = None
_c128 = np.ctypeslib.ndpointer(dtype=np.complex128, flags="C_CONTIGUOUS")
_f64 = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_i32 = np.ctypeslib.ndpointer(dtype=np.int32, flags="C_CONTIGUOUS")
_I, _D = ctypes.c_int, ctypes.c_double


def lib():
    global _lib
    if _lib is not None:
        return _lib
    L = ctypes.CDLL(build())
    L.cwo_oracle_set_threads.argtypes = [_I]
    L.cwo_oracle_get_threads.restype = _I
    L.cwo_oracle_max_threads.restype = _I
    L.cwo_oracle_dft1d.argtypes = [_I, _c128, _c128, _I]
    L.cwo_oracle_fft1d.argtypes = [_I, _c128, _c128, _I]
    L.cwo_oracle_fft2d.argtypes = [_I, _I, _c128, _I]
    L.cwo_oracle_dft2d.argtypes = [_I, _I, _c128, _c128, _I]
    L.cwo_oracle_asm_transfer.argtypes = [_I, _I, _D, _D, _D, _D, _c128]
    L.cwo_oracle_asm.argtypes = [_I, _I, _D, _D, _D, _D, _c128, _c128]
    L.cwo_oracle_asm_naive.argtypes = [_I, _I, _D, _D, _D, _D, _c128, _c128]
    L.cwo_oracle_asm_pad2x.argtypes = [_I, _I, _D, _D, _D, _D, _c128, _c128]
    L.cwo_oracle_stack.argtypes = [_I, _I, _D, _D, _D, _f64, _I, _c128, _c128]
    L.cwo_oracle_stack_intensity.argtypes = [_I, _I, _D, _D, _D, _f64, _I, _c128, _f64]
    L.cwo_oracle_asm_shifted.argtypes = [_I, _I, _D, _D, _D, _D, _D, _D, _c128, _c128]
    L.cwo_oracle_fresnel_points.argtypes = [_I, _I, _D, _D, _D, _D, _c128, _I, _i32, _i32, _c128]
    L.cwo_oracle_fresnel_direct.argtypes = [_I, _I, _D, _D, _D, _D, _c128, _c128]
    L.cwo_oracle_fresnel_conv.argtypes = [_I, _I, _D, _D, _D, _D, _c128, _c128]
    L.cwo_oracle_fresnel_general_direct.argtypes = [_I, _I, _f64, _D, _D, _c128, _c128]
    L.cwo_oracle_fresnel_general_points.argtypes = [_I, _I, _f64, _D, _D, _c128, _I, _i32, _i32, _c128]
    L.cwo_oracle_fresnel_fourier.argtypes = [_I, _I, _D, _D, _D, _D, _c128, _c128]
    L.cwo_oracle_fresnel_shifted.argtypes = [_I, _I, _f64, _D, _D, _c128, _c128]
    L.cwo_oracle_scale255.argtypes = [ctypes.c_size_t, _f64, _f64]
    L.cwo_oracle_pls_cgh.argtypes = [_I, _I, _D, _D, _D, _I, _f64, _f64, _f64, _f64, _f64]
    L.cwo_oracle_rs_direct.argtypes = [_I, _I, _D, _D, _D, _D, _c128, _c128]
    L.cwo_oracle_gs_init.argtypes = [_I, _I, _I, _D, _D, _D, _D, _f64, _f64, _c128]
    L.cwo_oracle_gs_iter.argtypes = [_I, _I, _I, _D, _D, _D, _D, _f64, _f64, _c128, ctypes.c_void_p]
    L.cwo_oracle_gs.argtypes = [_I, _I, _I, _D, _D, _D, _D, _I, _f64, _f64, _f64]
    L.cwo_oracle_gs_error.argtypes = [_I, _I, _I, _D, _D, _D, _D, _f64, _f64, _c128]
    L.cwo_oracle_gs_error.restype = _D
    _lib = L
    return L


def set_threads(t: int) -> None:
    lib().cwo_oracle_set_threads(int(t))


def max_threads() -> int:
    return int(lib().cwo_oracle_max_threads())


def _z(a) -> np.ndarray:
    """Widen (complex64-rounded) input to a fresh contiguous complex128 array."""
    return np.ascontiguousarray(a, dtype=np.complex128)


def _d(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def _check(rc: int, what: str) -> None:
    if rc != 0:
        raise ValueError("oracle %s failed with code %d" % (what, rc))


def dft1d(x, sign=-1):
    x = _z(x); out = np.empty_like(x)
    lib().cwo_oracle_dft1d(x.size, x, out, sign)
    return out


def fft1d(x, sign=-1):
    x = _z(x); out = np.empty_like(x)
    _check(lib().cwo_oracle_fft1d(x.size, x, out, sign), "fft1d")
    return out


def fft2d(a, sign=-1):
    a = _z(a).copy()
    ny, nx = a.shape
    _check(lib().cwo_oracle_fft2d(ny, nx, a, sign), "fft2d")
    return a


def dft2d(a, sign=-1):
    a = _z(a); out = np.empty_like(a)
    ny, nx = a.shape
    lib().cwo_oracle_dft2d(ny, nx, a, out, sign)
    return out


def asm_transfer(ny, nx, px, py, lam, z):
    H = np.empty((ny, nx), np.complex128)
    lib().cwo_oracle_asm_transfer(ny, nx, px, py, lam, z, H)
    return H


def asm(u1, px, py, lam, z, naive=False):
    """Angular spectrum method, Eq.(15)-(17) P:L194-211."""
    u1 = _z(u1); u2 = np.empty_like(u1)
    ny, nx = u1.shape
    if naive:
        lib().cwo_oracle_asm_naive(ny, nx, px, py, lam, z, u1, u2)
    else:
        _check(lib().cwo_oracle_asm(ny, nx, px, py, lam, z, u1, u2), "asm")
    return u2


def asm_pad2x(u1, px, py, lam, z):
    """ASM on the zero-expanded 2Nx x 2Ny grid, cropped (the paper's own form)."""
    u1 = _z(u1); u2 = np.empty_like(u1)
    ny, nx = u1.shape
    _check(lib().cwo_oracle_asm_pad2x(ny, nx, px, py, lam, z, u1, u2), "asm_pad2x")
    return u2


def stack(u1, px, py, lam, zs):
    """Diffract3D: out[k] = asm(u1, zs[k])."""
    u1 = _z(u1); zs = _d(zs)
    ny, nx = u1.shape
    out = np.empty((zs.size, ny, nx), np.complex128)
    _check(lib().cwo_oracle_stack(ny, nx, px, py, lam, zs, zs.size, u1, out), "stack")
    return out


def stack_intensity(u1, px, py, lam, zs):
    """|Diffract3D|^2, Eq.(20) P:L254-256 on every plane of the stack."""
    u1 = _z(u1); zs = _d(zs)
    ny, nx = u1.shape
    out = np.empty((zs.size, ny, nx), np.float64)
    _check(lib().cwo_oracle_stack_intensity(ny, nx, px, py, lam, zs, zs.size, u1, out), "stack_intensity")
    return out


def intensity(u):
    """Intensity of a complex amplitude, Eq.(20): I(m, n) = Re(u)^2 + Im(u)^2, in fp64 (the paper's c.Intensity()
    applied to one diffracted plane, Listing 1)."""
    u = _z(u)
    return u.real * u.real + u.imag * u.imag


def amplitude(u):
    """|u| = sqrt(re^2 + im^2): the "amplitude" real field of section 5, the square root of Eq.(20)."""
    return np.sqrt(intensity(u))


def re(u):
    """Real part of Eq.(24) P:L473-476 (the paper's Re(), conversion 1 P:L491)."""
    return _z(u).real.copy()


def im(u):
    """Imaginary part of Eq.(24) P:L473-476."""
    return _z(u).imag.copy()


def phase(u):
    """Argument of the complex amplitude, Eq.(25) P:L480-483 read as the four-quadrant atan2(im, re) in [-pi, pi] (the
    paper's Phase(), conversion 2 P:L497); 0 where u == 0 (phasor(0) = 1, as in the GS loop)."""
    u = _z(u)
    th = np.arctan2(u.imag, u.real)
    th[(u.real == 0) & (u.imag == 0)] = 0.0
    return th


def asm_shifted(u1, px, py, lam, z, ox=0.0, oy=0.0):
    """Shifted (band-limited) angular spectrum method, Eq.(18)-(19) P:L213-229; (ox, oy) = destination offset [m]."""
    u1 = _z(u1); u2 = np.empty_like(u1)
    ny, nx = u1.shape
    _check(lib().cwo_oracle_asm_shifted(ny, nx, px, py, lam, z, ox, oy, u1, u2), "asm_shifted")
    return u2


def fresnel_conv(u1, px, py, lam, z):
    """Literal Eq.(5) pipeline with the 2N expansion."""
    u1 = _z(u1); u2 = np.empty_like(u1)
    ny, nx = u1.shape
    _check(lib().cwo_oracle_fresnel_conv(ny, nx, px, py, lam, z, u1, u2), "fresnel_conv")
    return u2


def fresnel_direct(u1, px, py, lam, z):
    """Direct O(N^4) linear convolution = Eq.(1) discretised."""
    u1 = _z(u1); u2 = np.empty_like(u1)
    ny, nx = u1.shape
    lib().cwo_oracle_fresnel_direct(ny, nx, px, py, lam, z, u1, u2)
    return u2


def fresnel_points(u1, px, py, lam, z, ms, ns):
    """Direct-sum value of u2[ns[i], ms[i]] for a handful of samples (array indices)."""
    u1 = _z(u1)
    ny, nx = u1.shape
    ms = np.ascontiguousarray(ms, np.int32); ns = np.ascontiguousarray(ns, np.int32)
    out = np.empty(ms.size, np.complex128)
    lib().cwo_oracle_fresnel_points(ny, nx, px, py, lam, z, u1, ms.size, ms, ns, out)
    return out


def _geom(p0, p1, o0, o1):
    """(p0x, p0y, p1x, p1y, o0x, o0y, o1x, o1y): pitches [m] and lateral offsets [m] of the source / destination plane."""
    return np.array([p0[0], p0[1], p1[0], p1[1], o0[0], o0[1], o1[0], o1[1]], np.float64)


def fresnel_general_direct(u1, p0, p1, lam, z, o0=(0.0, 0.0), o1=(0.0, 0.0)):
    """Eq.(1) discretised between planes of pitch p0 / p1 = (px, py) and offsets o0 / o1 (direct O(N^4) sum)."""
    u1 = _z(u1); u2 = np.empty_like(u1)
    ny, nx = u1.shape
    lib().cwo_oracle_fresnel_general_direct(ny, nx, _geom(p0, p1, o0, o1), lam, z, u1, u2)
    return u2


def fresnel_general_points(u1, p0, p1, lam, z, ms, ns, o0=(0.0, 0.0), o1=(0.0, 0.0)):
    """Direct-sum value of u2[ns[i], ms[i]] (array indices) of the same sum, for full-size spot checks."""
    u1 = _z(u1)
    ny, nx = u1.shape
    ms = np.ascontiguousarray(ms, np.int32); ns = np.ascontiguousarray(ns, np.int32)
    out = np.empty(ms.size, np.complex128)
    lib().cwo_oracle_fresnel_general_points(ny, nx, _geom(p0, p1, o0, o1), lam, z, u1, ms.size, ms, ns, out)
    return out


def fresnel_fourier(u1, px, py, lam, z):
    """Fresnel diffraction, Fourier form, Eq.(7)-(9) P:L137-158; destination pitch lam |z| / (N p)."""
    u1 = _z(u1); u2 = np.empty_like(u1)
    ny, nx = u1.shape
    _check(lib().cwo_oracle_fresnel_fourier(ny, nx, px, py, lam, z, u1, u2), "fresnel_fourier")
    return u2


def fresnel_shifted(u1, p0, p1, lam, z, o0=(0.0, 0.0), o1=(0.0, 0.0)):
    """Shifted Fresnel diffraction, Eq.(10)-(14) P:L160-192."""
    u1 = _z(u1); u2 = np.empty_like(u1)
    ny, nx = u1.shape
    _check(lib().cwo_oracle_fresnel_shifted(ny, nx, _geom(p0, p1, o0, o1), lam, z, u1, u2), "fresnel_shifted")
    return u2


def scale255(a):
    """'Scale', Eq.(21) P:L258-262."""
    a = _d(a); out = np.empty_like(a)
    lib().cwo_oracle_scale255(a.size, a, out)
    return out


def pls_cgh(ny, nx, px, py, lam, xs, ys, zs, amps):
    """CGH of point light sources, Eq.(23) P:L327-332."""
    xs, ys, zs, amps = _d(xs), _d(ys), _d(zs), _d(amps)
    out = np.empty((ny, nx), np.float64)
    lib().cwo_oracle_pls_cgh(ny, nx, px, py, lam, xs.size, xs, ys, zs, amps, out)
    return out


def rs_direct(u1, px, py, lam, z):
    u1 = _z(u1); u2 = np.empty_like(u1)
    ny, nx = u1.shape
    lib().cwo_oracle_rs_direct(ny, nx, px, py, lam, z, u1, u2)
    return u2


def gs_init(method, amp_dst, phi0, px, py, lam, z):
    amp_dst = _d(amp_dst); phi0 = _d(phi0)
    ny, nx = amp_dst.shape
    p = np.empty((ny, nx), np.complex128)
    _check(lib().cwo_oracle_gs_init(method, ny, nx, px, py, lam, z, amp_dst, phi0, p), "gs_init")
    return p


def gs_iter(method, amp_src, amp_dst, p, px, py, lam, z, want_G=False):
    """One loop pass (Listing 8 lines 8-17).  Returns the new p (and G of this pass)."""
    amp_src = _d(amp_src); amp_dst = _d(amp_dst); p = _z(p).copy()
    ny, nx = p.shape
    G = np.empty_like(p) if want_G else None
    gp = G.ctypes.data_as(ctypes.c_void_p) if want_G else None
    _check(lib().cwo_oracle_gs_iter(method, ny, nx, px, py, lam, z, amp_src, amp_dst, p, gp), "gs_iter")
    return (p, G) if want_G else p


def gs(method, amp_src, amp_dst, phi0, px, py, lam, z, iters):
    amp_src = _d(amp_src); amp_dst = _d(amp_dst); ph = _d(phi0).copy()
    ny, nx = ph.shape
    _check(lib().cwo_oracle_gs(method, ny, nx, px, py, lam, z, iters, amp_src, amp_dst, ph), "gs")
    return ph


def gs_error(method, amp_src, amp_dst, p, px, py, lam, z):
    amp_src = _d(amp_src); amp_dst = _d(amp_dst); p = _z(p)
    ny, nx = p.shape
    return float(lib().cwo_oracle_gs_error(method, ny, nx, px, py, lam, z, amp_src, amp_dst, p))


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
