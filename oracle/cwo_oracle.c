/*
 * cwo_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, double-precision CPU statement of what the hot path of
 * arxiv/paper_1107_5578 (CWO++) computes.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load this file.
 * It shares no code, header, table or constant with the CUDA library
 * (paper_1107_5578_b200/csrc, include/cwo.h) and neither includes the other.
 *
 * Citations: P:Lnnn = /root/reference/PAPER.md line nnn; S8c = SURVEY.md section 8(c),
 * D-Rn = reading n in DESIGN.md ("Readings of the paper").
 *
 * Conventions (S8c, D-R3): forward DFT X[k] = sum_j x[j] exp(-i 2 pi j k / n),
 * inverse x[j] = (1/n) sum_k X[k] exp(+i 2 pi j k / n) -- the synthesis kernel
 * exp(+i 2 pi (fx x + fy y)) of Eq.(15) P:L198 with exp(+ikz) forward P:L102.
 * Fields are row-major [Ny][Nx], x fastest (interleaved re,im).
 *
 * Pin status (tests/test_oracle_*.py, all -m "not gpu"):
 *   fft1d / fft2d      pinned: naive DFT, Parseval, impulse<->constant, shift theorem
 *   asm                pinned: plane-wave eigenfunction vs 50-digit H, z=0 identity,
 *                              Parseval, semigroup, naive O(N^4) DFT brute force,
 *                              evanescent plane wave -> 0, Rayleigh-Sommerfeld sanity
 *   fresnel_conv       pinned: direct O(N^4) linear convolution, delta response closed
 *                              form, Gaussian-beam closed form, adjoint identity
 *   fresnel_point      pinned: equals fresnel_direct / closed forms (it IS Eq.(1) discretised)
 *   stack              pinned: equals n independent asm calls + semigroup
 *   stack_intensity    pinned: |stack|^2 element by element, sum = input energy (Parseval, no evanescent bin)
 *   asm_shifted        pinned: band covers the grid and O = 0 -> asm; plane wave inside the band -> H ramp u1 with
 *                              the band edge of Ref.[56]'s closed form typed in the test, outside -> exactly 0;
 *                              O = a whole number of pitches -> circular shift of asm (sign of the ramp);
 *                              z -> -z mirrors the band; the mask only removes energy
 *   fresnel_general_*  pinned: Gaussian-beam closed form sampled at another pitch and offset, delta response closed
 *                              form, equal pitches and no offset -> fresnel_direct (it IS Eq.(1) discretised)
 *   fresnel_fourier    pinned: fresnel_general_direct at the destination pitch lambda|z|/(N p) (both signs of z),
 *                              Gaussian-beam closed form, delta response closed form
 *   fresnel_shifted    pinned: fresnel_general_direct (pitches, offsets of both planes, z < 0), p1 = p0 and no offset
 *                              -> fresnel_conv, p1 = lambda z/(N p0) -> fresnel_fourier
 *   scale255           pinned: min -> 0, max -> 255, affine, numpy restatement
 *   pls_cgh            pinned: one on-axis point = Fresnel zone plate with zeros at the closed-form radii, symmetry,
 *                              linearity in A_j, numpy restatement at 50-digit-checked samples
 *   gs                 pinned: iters=0 kinoform identity, error non-increasing with the
 *                              unitary ASM propagator (Fienup), fixed point on a
 *                              consistent pair, step-by-step restatement in numpy
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double _Complex zc;

static const double TWO_PI = 6.283185307179586476925286766559;

/* ---- thread control (row/column parallelism only; arithmetic is unchanged) ---- */
static int g_threads = 1;
void cwo_oracle_set_threads(int t) { g_threads = t < 1 ? 1 : t; }
int  cwo_oracle_get_threads(void) { return g_threads; }
int  cwo_oracle_max_threads(void) {
#ifdef _OPENMP
    return omp_get_num_procs();
#else
    return 1;
#endif
}

/* exp(i 2 pi c) for c given in cycles; the integer part is removed first so the
 * argument of cos/sin stays in [0, 2 pi).  (Plain definition of a phase factor.) */
static zc cis_cycles(double c) {
    double f = c - floor(c);
    return cos(TWO_PI * f) + I * sin(TWO_PI * f);
}

/* ---- 1-D transforms ---------------------------------------------------------- */

/* Naive O(n^2) DFT, the definition itself.  sign = -1 forward, +1 inverse (with 1/n). */
void cwo_oracle_dft1d(int n, const zc* in, zc* out, int sign) {
    for (int k = 0; k < n; ++k) {
        zc acc = 0;
        for (int j = 0; j < n; ++j) {
            long long jk = ((long long)j * k) % n;          /* exact reduction of the angle */
            double a = TWO_PI * (double)jk / (double)n;
            acc += in[j] * (cos(a) + I * sign * sin(a));
        }
        out[k] = (sign > 0) ? acc / n : acc;
    }
}

/* Recursive radix-2 decimation in time.  tw[m] = exp(sign i 2 pi m / n0), m < n0/2,
 * each evaluated directly (no recurrence).  stride walks the input, step the table. */
static void fft_rec(int n, const zc* in, int stride, zc* out, const zc* tw, int step) {
    if (n == 1) { out[0] = in[0]; return; }
    int h = n / 2;
    fft_rec(h, in, 2 * stride, out, tw, 2 * step);               /* even samples */
    fft_rec(h, in + stride, 2 * stride, out + h, tw, 2 * step);  /* odd samples  */
    for (int k = 0; k < h; ++k) {
        zc e = out[k], o = tw[k * step] * out[k + h];
        out[k] = e + o;
        out[k + h] = e - o;
    }
}

/* Unnormalised radix-2 FFT with a caller-supplied table (n power of two). */
static void fft1d_tab(int n, const zc* in, zc* out, const zc* tw) { fft_rec(n, in, 1, out, tw, 1); }

static zc* make_twiddles(int n, int sign) {
    int h = n / 2 > 0 ? n / 2 : 1;
    zc* tw = (zc*)malloc(sizeof(zc) * h);
    for (int m = 0; m < h; ++m) {
        double a = TWO_PI * (double)m / (double)n;
        tw[m] = cos(a) + I * sign * sin(a);
    }
    return tw;
}

/* n must be a power of two.  sign = -1 forward, +1 inverse (with 1/n).  in != out. */
int cwo_oracle_fft1d(int n, const zc* in, zc* out, int sign) {
    if (n < 1 || (n & (n - 1))) return -1;
    zc* tw = make_twiddles(n, sign);
    fft1d_tab(n, in, out, tw);
    if (sign > 0) for (int k = 0; k < n; ++k) out[k] /= n;
    free(tw);
    return 0;
}

/* ---- 2-D transforms ---------------------------------------------------------- */

/* In-place 2-D FFT of a[ny][nx]: every row, then every column.  sign as above;
 * the inverse carries 1/(nx*ny) (D-R3). */
int cwo_oracle_fft2d(int ny, int nx, zc* a, int sign) {
    if (nx < 1 || ny < 1 || (nx & (nx - 1)) || (ny & (ny - 1))) return -1;
    zc* twx = make_twiddles(nx, sign);
    zc* twy = make_twiddles(ny, sign);
    #pragma omp parallel num_threads(g_threads)
    {
        int nmax = nx > ny ? nx : ny;
        zc* t0 = (zc*)malloc(sizeof(zc) * nmax);
        zc* t1 = (zc*)malloc(sizeof(zc) * nmax);
        #pragma omp for schedule(static)
        for (int y = 0; y < ny; ++y) {
            memcpy(t0, a + (size_t)y * nx, sizeof(zc) * nx);
            fft1d_tab(nx, t0, t1, twx);
            memcpy(a + (size_t)y * nx, t1, sizeof(zc) * nx);
        }
        #pragma omp for schedule(static)
        for (int x = 0; x < nx; ++x) {
            for (int y = 0; y < ny; ++y) t0[y] = a[(size_t)y * nx + x];
            fft1d_tab(ny, t0, t1, twy);
            for (int y = 0; y < ny; ++y) a[(size_t)y * nx + x] = t1[y];
        }
        free(t0); free(t1);
    }
    if (sign > 0) {
        double s = 1.0 / ((double)nx * (double)ny);
        for (size_t i = 0; i < (size_t)nx * ny; ++i) a[i] *= s;
    }
    free(twx); free(twy);
    return 0;
}

/* Naive O((nx ny)^2) 2-D DFT, out != in.  Tiny grids only. */
void cwo_oracle_dft2d(int ny, int nx, const zc* in, zc* out, int sign) {
    for (int l = 0; l < ny; ++l)
        for (int k = 0; k < nx; ++k) {
            zc acc = 0;
            for (int y = 0; y < ny; ++y)
                for (int x = 0; x < nx; ++x) {
                    double a = TWO_PI * ((double)(((long long)x * k) % nx) / nx +
                                         (double)(((long long)y * l) % ny) / ny);
                    acc += in[(size_t)y * nx + x] * (cos(a) + I * sign * sin(a));
                }
            out[(size_t)l * nx + k] = (sign > 0) ? acc / ((double)nx * ny) : acc;
        }
}

/* ---- angular spectrum method: Eq.(15)-(17), P:L194-211 ----------------------- */

/* FFT-order signed bin: k < n/2 -> k, else k - n (S8c; the Nyquist bin is negative). */
static double signed_bin(int k, int n) { return (double)((k < n / 2) ? k : k - n); }

/* H_A(k,l) of Eq.(16) P:L203 written with 1/lambda: z sqrt(k^2 - 4 pi^2 f^2) = 2 pi z sqrt(1/lambda^2 - f^2).
 * w < 0 (evanescent) -> 0 (north_star, D-R2); w == 0 propagates.  The expression for w is the one
 * S8c/A4 fixes: inv_lam2 - (fx*fx + fy*fy). */
static zc asm_H(int k, int l, int nx, int ny, double px, double py, double lambda, double z) {
    double dfx = 1.0 / ((double)nx * px), dfy = 1.0 / ((double)ny * py);
    double fx = signed_bin(k, nx) * dfx, fy = signed_bin(l, ny) * dfy;
    double inv_lam2 = 1.0 / (lambda * lambda);
    double w = inv_lam2 - (fx * fx + fy * fy);
    if (w < 0.0) return 0;
    return cis_cycles(z * sqrt(w));
}

void cwo_oracle_asm_transfer(int ny, int nx, double px, double py, double lambda, double z, zc* H) {
    for (int l = 0; l < ny; ++l)
        for (int k = 0; k < nx; ++k) H[(size_t)l * nx + k] = asm_H(k, l, nx, ny, px, py, lambda, z);
}

/* u2 = IDFT2[ DFT2[u1] . H ]  (Eq.(17)), unpadded N x N circular (D-R1). */
int cwo_oracle_asm(int ny, int nx, double px, double py, double lambda, double z, const zc* u1, zc* u2) {
    size_t n = (size_t)nx * ny;
    if (u2 != u1) memcpy(u2, u1, sizeof(zc) * n);
    if (cwo_oracle_fft2d(ny, nx, u2, -1)) return -1;
    #pragma omp parallel for num_threads(g_threads) schedule(static)
    for (int l = 0; l < ny; ++l)
        for (int k = 0; k < nx; ++k) u2[(size_t)l * nx + k] *= asm_H(k, l, nx, ny, px, py, lambda, z);
    return cwo_oracle_fft2d(ny, nx, u2, +1);
}

/* Same definition with the two DFTs evaluated naively (O(N^4)); tiny grids. */
void cwo_oracle_asm_naive(int ny, int nx, double px, double py, double lambda, double z, const zc* u1, zc* u2) {
    size_t n = (size_t)nx * ny;
    zc* A = (zc*)malloc(sizeof(zc) * n);
    cwo_oracle_dft2d(ny, nx, u1, A, -1);
    for (int l = 0; l < ny; ++l)
        for (int k = 0; k < nx; ++k) A[(size_t)l * nx + k] *= asm_H(k, l, nx, ny, px, py, lambda, z);
    cwo_oracle_dft2d(ny, nx, A, u2, +1);
    free(A);
}

/* the paper's own form of ASM: like every "convolution form" method it expands the calculation
 * area to 2Nx x 2Ny with zeros to avoid the wrap-around of the circular convolution (Table 2
 * P:L287-289).  u1 sits in the [0,Ny) x [0,Nx) corner of the zero array, Eq.(15)-(17) run on the 2N grid
 * (so the frequency sampling is 1/(2 N p)), and the same corner is cropped.  The convolution is shift
 * invariant, so the result does not depend on where in the big array the window sits. */
int cwo_oracle_asm_pad2x(int ny, int nx, double px, double py, double lambda, double z, const zc* u1, zc* u2) {
    int my = 2 * ny, mx = 2 * nx;
    zc* a = (zc*)calloc((size_t)mx * my, sizeof(zc));
    if (!a) return -1;
    for (int r = 0; r < ny; ++r) memcpy(a + (size_t)r * mx, u1 + (size_t)r * nx, sizeof(zc) * nx);
    int rc = cwo_oracle_asm(my, mx, px, py, lambda, z, a, a);
    if (!rc) for (int r = 0; r < ny; ++r) memcpy(u2 + (size_t)r * nx, a + (size_t)r * mx, sizeof(zc) * nx);
    free(a);
    return rc;
}

/* 3-D diffraction = 2-D diffractions stacked along z (Listing 2):
 * out[k] = asm(u1, zs[k]).  Written as n independent calls on purpose. */
int cwo_oracle_stack(int ny, int nx, double px, double py, double lambda, const double* zs, int n,
                     const zc* u1, zc* out) {
    for (int k = 0; k < n; ++k)
        if (cwo_oracle_asm(ny, nx, px, py, lambda, zs[k], u1, out + (size_t)k * nx * ny)) return -1;
    return 0;
}

/* Intensity of every plane of the stack, Eq.(20): I = |u|^2 (what the paper's 3-D example stores for
 * rendering).  Written as the stack followed by the absolute square. */
int cwo_oracle_stack_intensity(int ny, int nx, double px, double py, double lambda, const double* zs, int n,
                               const zc* u1, double* out) {
    size_t f = (size_t)nx * ny;
    zc* plane = (zc*)malloc(sizeof(zc) * f);
    if (!plane) return -1;
    for (int k = 0; k < n; ++k) {
        if (cwo_oracle_asm(ny, nx, px, py, lambda, zs[k], u1, plane)) { free(plane); return -1; }
        for (size_t i = 0; i < f; ++i) {
            double re = creal(plane[i]), im = cimag(plane[i]);
            out[(size_t)k * f + i] = re * re + im * im;
        }
    }
    free(plane);
    return 0;
}

/* ---- shifted (band-limited) angular spectrum method: Eq.(18)-(19), P:L213-229 ---------------------------------
 * u2 = IDFT2[ DFT2[u1] . H_SA . Rect((m1-cx)/wx) . Rect((n1-cy)/wy) ],
 * H_SA = H_A exp(i 2 pi (Ox fx + Oy fy))                  (Eq.(19); the "i" is missing in the extracted text, D-R15)
 * The paper refers to its Ref.[56] for cx, wx, cy, wy.  D-R15: they are the bins where the phase of H_SA,
 * sampled at the pitch df of the frequency grid, is not aliased -- its local frequency |d(phase)/df| / 2 pi =
 * |O - z f / sqrt(1/lambda^2 - f^2)| must not exceed 1/(2 df) -- evaluated per axis ON that axis (the other
 * frequency 0), which is what makes the limit a product of two Rects.  A bin with f^2 >= 1/lambda^2 is outside. */
static int shifted_keep(double f, double df, double off, double lambda, double z) {
    double inv_lam2 = 1.0 / (lambda * lambda);
    double w = inv_lam2 - f * f;
    if (w <= 0.0) return 0;
    return fabs(off - z * f / sqrt(w)) <= 0.5 / df;
}

int cwo_oracle_asm_shifted(int ny, int nx, double px, double py, double lambda, double z, double ox, double oy,
                           const zc* u1, zc* u2) {
    size_t n = (size_t)nx * ny;
    double dfx = 1.0 / ((double)nx * px), dfy = 1.0 / ((double)ny * py);
    if (u2 != u1) memcpy(u2, u1, sizeof(zc) * n);
    if (cwo_oracle_fft2d(ny, nx, u2, -1)) return -1;
    #pragma omp parallel for num_threads(g_threads) schedule(static)
    for (int l = 0; l < ny; ++l)
        for (int k = 0; k < nx; ++k) {
            double fx = signed_bin(k, nx) * dfx, fy = signed_bin(l, ny) * dfy;
            zc h = 0;
            if (shifted_keep(fx, dfx, ox, lambda, z) && shifted_keep(fy, dfy, oy, lambda, z))
                h = asm_H(k, l, nx, ny, px, py, lambda, z) * cis_cycles(ox * fx + oy * fy);
            u2[(size_t)l * nx + k] *= h;
        }
    return cwo_oracle_fft2d(ny, nx, u2, +1);
}

/* ---- Fresnel diffraction, convolution form: Eq.(1)-(6), P:L98-135 ------------ */

/* h_F of Eq.(3)/(6) P:L113, P:L132 (the garbled "pi/4tau" read as pi/(lambda z), D-R5) at the
 * integer offset (dm, dn): exp(i pi ((dm px)^2 + (dn py)^2) / (lambda z)). */
static zc fresnel_h(int dm, int dn, double px, double py, double lambda, double z) {
    double x = dm * px, y = dn * py;
    return cis_cycles((x * x + y * y) / (2.0 * lambda * z));
}

/* exp(i 2 pi z / lambda) / (i lambda z) * px * py: the prefactor of Eq.(1) P:L102 times the area
 * element of the discretised integral (D-R6). */
static zc fresnel_coeff(double px, double py, double lambda, double z) {
    return cis_cycles(z / lambda) / (I * lambda * z) * (px * py);
}

/* One output sample of Eq.(1) discretised on the N x N window (plain definition = direct
 * linear convolution, S8c O-FRES): u2[n2][m2] = c * sum u1[n1][m1] h_F(m2-m1, n2-n1). */
static zc fresnel_point_value(int ny, int nx, double px, double py, double lambda, double z,
                                  const zc* u1, int m2, int n2) {
    zc acc = 0;
    for (int n1 = 0; n1 < ny; ++n1) {
        zc row = 0;
        for (int m1 = 0; m1 < nx; ++m1) {
            zc v = u1[(size_t)n1 * nx + m1];
            if (v != 0) row += v * fresnel_h(m2 - m1, n2 - n1, px, py, lambda, z);
        }
        acc += row;
    }
    return fresnel_coeff(px, py, lambda, z) * acc;
}

/* Samples (ms[i], ns[i]) of the direct sum; used for full-size spot checks. */
void cwo_oracle_fresnel_points(int ny, int nx, double px, double py, double lambda, double z,
                               const zc* u1, int npts, const int* ms, const int* ns, zc* out) {
    #pragma omp parallel for num_threads(g_threads) schedule(dynamic, 1)
    for (int i = 0; i < npts; ++i)
        out[i] = fresnel_point_value(ny, nx, px, py, lambda, z, u1, ms[i], ns[i]);
}

/* Whole-field direct sum, O(N^4).  Tiny grids. */
void cwo_oracle_fresnel_direct(int ny, int nx, double px, double py, double lambda, double z,
                               const zc* u1, zc* u2) {
    #pragma omp parallel for num_threads(g_threads) schedule(static)
    for (int n2 = 0; n2 < ny; ++n2)
        for (int m2 = 0; m2 < nx; ++m2)
            u2[(size_t)n2 * nx + m2] =
                fresnel_point_value(ny, nx, px, py, lambda, z, u1, m2, n2);
}

/* The literal Eq.(5) pipeline with the 2Nx x 2Ny expansion of P:L235:
 * pad u1 into the [0,N) corner of a zero 2N x 2N array; sample h_F at taps d = -N..N-1 per
 * axis stored wrapped at index d mod 2N; FFT2 both; multiply; IFFT2; keep [0,N); times the
 * coefficient.  Where u1 sits in the padded array does not change the cropped result (D-R7). */
int cwo_oracle_fresnel_conv(int ny, int nx, double px, double py, double lambda, double z,
                            const zc* u1, zc* u2) {
    if (z == 0.0) return -2;                                   /* 1/(i lambda z) singular (D-R8) */
    int mx = 2 * nx, my = 2 * ny;
    size_t mm = (size_t)mx * my;
    zc* U = (zc*)calloc(mm, sizeof(zc));
    zc* Hh = (zc*)malloc(sizeof(zc) * mm);
    if (!U || !Hh) { free(U); free(Hh); return -3; }
    for (int y = 0; y < ny; ++y) memcpy(U + (size_t)y * mx, u1 + (size_t)y * nx, sizeof(zc) * nx);
    #pragma omp parallel for num_threads(g_threads) schedule(static)
    for (int iy = 0; iy < my; ++iy) {
        int dn = (iy < ny) ? iy : iy - my;
        for (int ix = 0; ix < mx; ++ix) {
            int dm = (ix < nx) ? ix : ix - mx;
            Hh[(size_t)iy * mx + ix] = fresnel_h(dm, dn, px, py, lambda, z);
        }
    }
    int rc = cwo_oracle_fft2d(my, mx, U, -1);
    if (!rc) rc = cwo_oracle_fft2d(my, mx, Hh, -1);
    if (!rc) {
        for (size_t i = 0; i < mm; ++i) U[i] *= Hh[i];
        rc = cwo_oracle_fft2d(my, mx, U, +1);
    }
    if (!rc) {
        zc c = fresnel_coeff(px, py, lambda, z);
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) u2[(size_t)y * nx + x] = c * U[(size_t)y * mx + x];
    }
    free(U); free(Hh);
    return rc;
}

/* ---- Fresnel diffraction between planes of different pitch and lateral offset ------------------
 * Eq.(1) P:L102 discretised with the source plane sampled at x0 = m0 p0x + O0x and the destination at
 * x1 = m1 p1x + O1x (Eq.(14)), m = array index - N/2 (Eq.(4)):
 *   u2[n1][m1] = exp(i 2 pi z/lambda)/(i lambda z) p0x p0y sum_{m0,n0} u1[n0][m0]
 *                exp(i pi ((x1 - x0)^2 + (y1 - y0)^2)/(lambda z)).
 * This sum is what BOTH the Fourier form (Eq.(7)-(9) P:L137-158) and the shifted Fresnel diffraction
 * (Eq.(10)-(14) P:L160-192) evaluate; it is their plain definition (area element as in D-R6).
 * Offsets are in metres (D-R16: the paper's O are in samples of their own plane, O[m] = p O[samples]). */
typedef struct { double p0x, p0y, p1x, p1y, o0x, o0y, o1x, o1y; } fres_geom;

static zc fresnel_general_point(int ny, int nx, const fres_geom* g, double lambda, double z,
                                const zc* u1, int m1i, int n1i) {
    double x1 = (m1i - nx / 2) * g->p1x + g->o1x, y1 = (n1i - ny / 2) * g->p1y + g->o1y;
    zc acc = 0;
    for (int n0 = 0; n0 < ny; ++n0) {
        double dy = y1 - ((n0 - ny / 2) * g->p0y + g->o0y);
        zc row = 0;
        for (int m0 = 0; m0 < nx; ++m0) {
            zc v = u1[(size_t)n0 * nx + m0];
            if (v == 0) continue;
            double dx = x1 - ((m0 - nx / 2) * g->p0x + g->o0x);
            row += v * cis_cycles((dx * dx + dy * dy) / (2.0 * lambda * z));
        }
        acc += row;
    }
    return fresnel_coeff(g->p0x, g->p0y, lambda, z) * acc;
}

/* Whole field by the direct sum, O(N^4): tiny grids.  geom = {p0x,p0y,p1x,p1y,o0x,o0y,o1x,o1y}. */
void cwo_oracle_fresnel_general_direct(int ny, int nx, const double* geom, double lambda, double z,
                                       const zc* u1, zc* u2) {
    fres_geom g = {geom[0], geom[1], geom[2], geom[3], geom[4], geom[5], geom[6], geom[7]};
    #pragma omp parallel for num_threads(g_threads) schedule(static)
    for (int n1 = 0; n1 < ny; ++n1)
        for (int m1 = 0; m1 < nx; ++m1)
            u2[(size_t)n1 * nx + m1] = fresnel_general_point(ny, nx, &g, lambda, z, u1, m1, n1);
}

/* Samples (ms[i], ns[i]) (array indices) of the direct sum, for full-size spot checks. */
void cwo_oracle_fresnel_general_points(int ny, int nx, const double* geom, double lambda, double z,
                                       const zc* u1, int npts, const int* ms, const int* ns, zc* out) {
    fres_geom g = {geom[0], geom[1], geom[2], geom[3], geom[4], geom[5], geom[6], geom[7]};
    #pragma omp parallel for num_threads(g_threads) schedule(dynamic, 1)
    for (int i = 0; i < npts; ++i)
        out[i] = fresnel_general_point(ny, nx, &g, lambda, z, u1, ms[i], ns[i]);
}

/* Fresnel diffraction, Fourier form, the literal Eq.(8)-(9) P:L149-156:
 *   u' = u1 exp(i pi (x1^2 + y1^2)/(lambda z));   U = FFT[u'] over the centred indices m = j - N/2;
 *   u2 = exp(i 2 pi z/lambda)/(i lambda z) exp(i pi (x2^2 + y2^2)/(lambda z)) U  (times p1x p1y, D-R6),
 * on the destination pitch p2 = lambda |z| / (N p1) (D-R17: P:L158's "Delta x1/(lambda z)" is garbled; this is the
 * pitch at which the kernel exp(-i 2 pi x2 x1/(lambda z)) of Eq.(7) becomes the DFT kernel exp(-+ i 2 pi m1 m2/N);
 * for z < 0 its sign flips and "FFT" is the unnormalised inverse transform).  The centred transform is taken by
 * rotating the array by N/2 before and after a plain FFT (the DFT kernel is periodic in both indices). */
int cwo_oracle_fresnel_fourier(int ny, int nx, double px, double py, double lambda, double z,
                               const zc* u1, zc* u2) {
    if (z == 0.0) return -2;
    if (nx < 2 || ny < 2 || (nx & (nx - 1)) || (ny & (ny - 1))) return -1;
    size_t n = (size_t)nx * ny;
    double p2x = lambda * fabs(z) / (nx * px), p2y = lambda * fabs(z) / (ny * py);
    zc* a = (zc*)malloc(sizeof(zc) * n);
    if (!a) return -3;
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            double x = (i - nx / 2) * px, y = (j - ny / 2) * py;
            zc v = u1[(size_t)j * nx + i] * cis_cycles((x * x + y * y) / (2.0 * lambda * z));      /* Eq.(8) */
            a[(size_t)((j + ny / 2) % ny) * nx + (i + nx / 2) % nx] = v;                          /* m = 0 -> index 0 */
        }
    int rc = cwo_oracle_fft2d(ny, nx, a, z > 0 ? -1 : +1);
    if (!rc) {
        double undo = z > 0 ? 1.0 : (double)nx * (double)ny;       /* fft2d's inverse carries 1/(nx ny); Eq.(9) does not */
        zc c = fresnel_coeff(px, py, lambda, z);
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                double x = (i - nx / 2) * p2x, y = (j - ny / 2) * p2y;
                zc U = a[(size_t)((j + ny / 2) % ny) * nx + (i + nx / 2) % nx] * undo;
                u2[(size_t)j * nx + i] = c * cis_cycles((x * x + y * y) / (2.0 * lambda * z)) * U;  /* Eq.(9) */
            }
    }
    free(a);
    return rc;
}

/* Shifted Fresnel diffraction, the algorithm of Eq.(10)-(14) P:L160-192 step by step (paper's notation, plane 0 =
 * source, plane 1 = destination; S = p0 p1/(lambda z)):
 *   u1'[m0,n0] = u1 exp(i pi (x0^2 + y0^2)/(lambda z)) exp(-i 2 pi (m0 Sx O1x/p1x + n0 Sy O1y/p1y))
 *                exp(-i pi (Sx m0^2 + Sy n0^2))                                                   Eq.(12)
 *   h[m,n]     = exp(i pi (Sx m^2 + Sy n^2))                                                      Eq.(13)
 *   C_S[m1,n1] = coefficient exp(i pi (x1^2 + y1^2)/(lambda z)) exp(-i 2 pi (O0x x1 + O0y y1)/(lambda z))
 *                exp(-i pi (Sx m1^2 + Sy n1^2))                                                   Eq.(11)
 *   u2 = C_S IFFT[FFT[u1'] FFT[h]]                                                                Eq.(10)
 * with the convolution made linear by the 2N expansion of P:L235 exactly as in fresnel_conv (taps d = -N..N-1
 * wrapped at d mod 2N).  m, n are the centred indices; the coefficient carries p0x p0y (D-R6). */
int cwo_oracle_fresnel_shifted(int ny, int nx, const double* geom, double lambda, double z,
                               const zc* u1, zc* u2) {
    if (z == 0.0) return -2;
    fres_geom g = {geom[0], geom[1], geom[2], geom[3], geom[4], geom[5], geom[6], geom[7]};
    const double sx = g.p0x * g.p1x / (lambda * z), sy = g.p0y * g.p1y / (lambda * z);
    int mx = 2 * nx, my = 2 * ny;
    size_t mm = (size_t)mx * my;
    zc* U = (zc*)calloc(mm, sizeof(zc));
    zc* Hh = (zc*)malloc(sizeof(zc) * mm);
    if (!U || !Hh) { free(U); free(Hh); return -3; }
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            double m0 = i - nx / 2, n0 = j - ny / 2;
            double x0 = m0 * g.p0x + g.o0x, y0 = n0 * g.p0y + g.o0y;
            zc f = cis_cycles((x0 * x0 + y0 * y0) / (2.0 * lambda * z))
                 * cis_cycles(-(m0 * sx * g.o1x / g.p1x + n0 * sy * g.o1y / g.p1y))
                 * cis_cycles(-0.5 * (sx * m0 * m0 + sy * n0 * n0));
            U[(size_t)j * mx + i] = u1[(size_t)j * nx + i] * f;                                   /* Eq.(12) */
        }
    #pragma omp parallel for num_threads(g_threads) schedule(static)
    for (int iy = 0; iy < my; ++iy) {
        double dn = (iy < ny) ? iy : iy - my;
        for (int ix = 0; ix < mx; ++ix) {
            double dm = (ix < nx) ? ix : ix - mx;
            Hh[(size_t)iy * mx + ix] = cis_cycles(0.5 * (sx * dm * dm + sy * dn * dn));           /* Eq.(13) */
        }
    }
    int rc = cwo_oracle_fft2d(my, mx, U, -1);
    if (!rc) rc = cwo_oracle_fft2d(my, mx, Hh, -1);
    if (!rc) {
        for (size_t i = 0; i < mm; ++i) U[i] *= Hh[i];
        rc = cwo_oracle_fft2d(my, mx, U, +1);                                                      /* Eq.(10) */
    }
    if (!rc) {
        zc c = fresnel_coeff(g.p0x, g.p0y, lambda, z);
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                double m1 = i - nx / 2, n1 = j - ny / 2;
                double x1 = m1 * g.p1x + g.o1x, y1 = n1 * g.p1y + g.o1y;
                zc cs = c * cis_cycles((x1 * x1 + y1 * y1) / (2.0 * lambda * z))
                          * cis_cycles(-(g.o0x * x1 + g.o0y * y1) / (lambda * z))
                          * cis_cycles(-0.5 * (sx * m1 * m1 + sy * n1 * n1));                      /* Eq.(11) */
                u2[(size_t)j * nx + i] = cs * U[(size_t)j * mx + i];
            }
    }
    free(U); free(Hh);
    return rc;
}

/* ---- output conversions of Listings 1-3 ------------------------------------------------------- */

/* "Scale", Eq.(21): I256 = (I - min I)/(max I - min I) * 255 (a constant field maps to 0, D-R18). */
void cwo_oracle_scale255(size_t n, const double* in, double* out) {
    double lo = in[0], hi = in[0];
    for (size_t i = 1; i < n; ++i) { if (in[i] < lo) lo = in[i]; if (in[i] > hi) hi = in[i]; }
    for (size_t i = 0; i < n; ++i) out[i] = (hi > lo) ? (in[i] - lo) / (hi - lo) * 255.0 : 0.0;
}

/* CGH from point light sources, Eq.(23) P:L327-332:
 *   I(x, y) = sum_j A_j cos( (2 pi/lambda) ((x - x_j)^2 + (y - y_j)^2)/(2 z_j) ),
 * (x, y) = ((i - nx/2) px, (j - ny/2) py) on the hologram (Eq.(4)). */
void cwo_oracle_pls_cgh(int ny, int nx, double px, double py, double lambda, int npts,
                        const double* xs, const double* ys, const double* zs, const double* amps, double* out) {
    #pragma omp parallel for num_threads(g_threads) schedule(static)
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            double x = (i - nx / 2) * px, y = (j - ny / 2) * py, acc = 0.0;
            for (int k = 0; k < npts; ++k) {
                double dx = x - xs[k], dy = y - ys[k];
                double c = (dx * dx + dy * dy) / (2.0 * lambda * zs[k]);     /* cycles */
                acc += amps[k] * cos(TWO_PI * (c - floor(c)));
            }
            out[(size_t)j * nx + i] = acc;
        }
}

/* ---- Rayleigh-Sommerfeld I quadrature (Goodman, ref [1] P:L765) -- sanity only -- */
/* u2 = (1/2pi) sum u1 (z/r)(1/r - ik) exp(ikr)/r px py,  r = sqrt(z^2 + dx^2 + dy^2). */
void cwo_oracle_rs_direct(int ny, int nx, double px, double py, double lambda, double z,
                          const zc* u1, zc* u2) {
    double k = TWO_PI / lambda;
    #pragma omp parallel for num_threads(g_threads) schedule(static)
    for (int n2 = 0; n2 < ny; ++n2)
        for (int m2 = 0; m2 < nx; ++m2) {
            zc acc = 0;
            for (int n1 = 0; n1 < ny; ++n1)
                for (int m1 = 0; m1 < nx; ++m1) {
                    double dx = (m2 - m1) * px, dy = (n2 - n1) * py;
                    double r = sqrt(z * z + dx * dx + dy * dy);
                    acc += u1[(size_t)n1 * nx + m1] * ((z / r) * (1.0 / r - I * k)) *
                           cis_cycles(r / lambda) / r;
                }
            u2[(size_t)n2 * nx + m2] = acc * (px * py) / TWO_PI;
        }
}

/* ---- Gerchberg-Saxton: Listing 8 P:L687-709 (S8c O-GS, D-R9..R12) -- */

/* phasor(u) = u/|u|, 1 where |u| = 0 (atan2(0,0) = 0, Eq.(25)). */
static zc phasor(zc u) {
    double a = cabs(u);
    return (a == 0.0) ? 1.0 : u / a;
}

/* P(z): method 0 = Fresnel convolution (config c5), 1 = angular spectrum (paper's Listing 8). */
static int gs_prop(int method, int ny, int nx, double px, double py, double lambda, double z,
                   const zc* in, zc* out) {
    return method ? cwo_oracle_asm(ny, nx, px, py, lambda, z, in, out)
                  : cwo_oracle_fresnel_conv(ny, nx, px, py, lambda, z, in, out);
}

/* Step 1-2 (Listing 8 lines 3-7): G = amp_dst exp(i phi0); p = phasor(P(-z)[G]). */
int cwo_oracle_gs_init(int method, int ny, int nx, double px, double py, double lambda, double z,
                       const double* amp_dst, const double* phi0, zc* p) {
    size_t n = (size_t)nx * ny;
    zc* G = (zc*)malloc(sizeof(zc) * n);
    for (size_t i = 0; i < n; ++i) G[i] = amp_dst[i] * (cos(phi0[i]) + I * sin(phi0[i]));
    int rc = gs_prop(method, ny, nx, px, py, lambda, -z, G, p);
    for (size_t i = 0; i < n; ++i) p[i] = phasor(p[i]);
    free(G);
    return rc;
}

/* Step 3, one pass of the loop (Listing 8 lines 8-17):
 *   G = P(+z)[amp_src . p];  q = phasor(G);  p = phasor(P(-z)[amp_dst . q]).
 * G_out (optional) receives the reconstruction G of this iteration (for the error metric). */
int cwo_oracle_gs_iter(int method, int ny, int nx, double px, double py, double lambda, double z,
                       const double* amp_src, const double* amp_dst, zc* p, zc* G_out) {
    size_t n = (size_t)nx * ny;
    zc* a = (zc*)malloc(sizeof(zc) * n);
    zc* G = (zc*)malloc(sizeof(zc) * n);
    for (size_t i = 0; i < n; ++i) a[i] = amp_src[i] * p[i];
    int rc = gs_prop(method, ny, nx, px, py, lambda, z, a, G);
    if (G_out) memcpy(G_out, G, sizeof(zc) * n);
    for (size_t i = 0; i < n; ++i) a[i] = amp_dst[i] * phasor(G[i]);
    if (!rc) rc = gs_prop(method, ny, nx, px, py, lambda, -z, a, p);
    for (size_t i = 0; i < n; ++i) p[i] = phasor(p[i]);
    free(a); free(G);
    return rc;
}

/* Whole call: phase (in: phi0, out: atan2(Im p, Re p) in (-pi, pi]).  2*iters+1 propagations. */
int cwo_oracle_gs(int method, int ny, int nx, double px, double py, double lambda, double z, int iters,
                  const double* amp_src, const double* amp_dst, double* phase) {
    size_t n = (size_t)nx * ny;
    zc* p = (zc*)malloc(sizeof(zc) * n);
    int rc = cwo_oracle_gs_init(method, ny, nx, px, py, lambda, z, amp_dst, phase, p);
    for (int t = 0; t < iters && !rc; ++t)
        rc = cwo_oracle_gs_iter(method, ny, nx, px, py, lambda, z, amp_src, amp_dst, p, NULL);
    for (size_t i = 0; i < n; ++i) phase[i] = atan2(cimag(p[i]), creal(p[i]));
    free(p);
    return rc;
}

/* eps = || |P(+z)[amp_src . p]| - amp_dst || / || amp_dst ||  (S8c G5 (ii)). */
double cwo_oracle_gs_error(int method, int ny, int nx, double px, double py, double lambda, double z,
                           const double* amp_src, const double* amp_dst, const zc* p) {
    size_t n = (size_t)nx * ny;
    zc* a = (zc*)malloc(sizeof(zc) * n);
    zc* G = (zc*)malloc(sizeof(zc) * n);
    for (size_t i = 0; i < n; ++i) a[i] = amp_src[i] * p[i];
    gs_prop(method, ny, nx, px, py, lambda, z, a, G);
    double num = 0, den = 0;
    for (size_t i = 0; i < n; ++i) {
        double d = cabs(G[i]) - amp_dst[i];
        num += d * d; den += amp_dst[i] * amp_dst[i];
    }
    free(a); free(G);
    return sqrt(num / den);
}
