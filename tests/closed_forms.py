"""Closed forms of the paper's formulas evaluated in 50-digit arithmetic (mpmath).

Independent of oracle/ (C, double) and of the CUDA path: used to pin both.
  asm_H      Eq.(16):  H = exp(i z sqrt(k^2 - 4 pi^2 (fx^2+fy^2))),  f = bin / (N pitch)
  fresnel_delta   Eq.(1) P:L102 on a single source sample: c * h_F(offset), h_F of Eq.(3) P:L113,
                  c = exp(i 2 pi z / lambda) / (i lambda z) * px * py  (area element: DESIGN.md reading R6)
  gaussian_beam   Fresnel propagation of exp(-r^2/w0^2): exp(ikz) (1/q) exp(-r^2/(w0^2 q)), q = 1 + i z/z_R
Decimal strings keep lambda, pitch, z exact ("633e-9" is not a double).
"""
from mpmath import mp, mpf, sqrt, floor, exp, pi

mp.dps = 50


def _m(v):
    return mpf(v) if isinstance(v, str) else mpf(repr(float(v)))


def asm_cycles(nx, ny, px, py, lam, z, k, l):
    px, py, lam, z = _m(px), _m(py), _m(lam), _m(z)
    fx = mpf(k) / (nx * px); fy = mpf(l) / (ny * py)
    w = 1 / lam ** 2 - fx ** 2 - fy ** 2
    return None if w < 0 else z * sqrt(w)


def asm_H(nx, ny, px, py, lam, z, k, l):
    c = asm_cycles(nx, ny, px, py, lam, z, k, l)
    if c is None:
        return 0j
    return complex(exp(2j * pi * (c - floor(c))))


def fresnel_delta(px, py, lam, z, dm, dn):
    px, py, lam, z = _m(px), _m(py), _m(lam), _m(z)
    c = exp(2j * pi * (z / lam - floor(z / lam))) / (1j * lam * z) * px * py
    ph = ((dm * px) ** 2 + (dn * py) ** 2) / (2 * lam * z)
    return complex(c * exp(2j * pi * (ph - floor(ph))))


def gaussian_beam(lam, z, w0, x, y):
    lam, z, w0, x, y = _m(lam), _m(z), _m(w0), _m(x), _m(y)
    zR = pi * w0 ** 2 / lam
    q = 1 + 1j * z / zR
    return complex(exp(2j * pi * (z / lam - floor(z / lam))) / q * exp(-(x * x + y * y) / (w0 ** 2 * q)))


def fresnel_delta_xy(p0x, p0y, lam, z, dx, dy):
    """Eq.(1) P:L102 on one source sample seen from a point (dx, dy) metres away laterally:
    exp(i 2 pi z/lambda)/(i lambda z) p0x p0y exp(i pi (dx^2 + dy^2)/(lambda z))."""
    p0x, p0y, lam, z, dx, dy = _m(p0x), _m(p0y), _m(lam), _m(z), _m(dx), _m(dy)
    c = exp(2j * pi * (z / lam - floor(z / lam))) / (1j * lam * z) * p0x * p0y
    ph = (dx * dx + dy * dy) / (2 * lam * z)
    return complex(c * exp(2j * pi * (ph - floor(ph))))


def pls_term(lam, zj, dx, dy):
    """One term of Eq.(23) P:L327-332 with A_j = 1: cos((2 pi/lambda) (dx^2 + dy^2)/(2 zj))."""
    from mpmath import cos
    lam, zj, dx, dy = _m(lam), _m(zj), _m(dx), _m(dy)
    ph = (dx * dx + dy * dy) / (2 * lam * zj)
    return float(cos(2 * pi * (ph - floor(ph))))
