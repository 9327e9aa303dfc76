// tables.cu -- small double-precision table builders.
//   * FFT twiddles exp(-i 2 pi m/n), evaluated in fp64 and rounded once to fp32.
//   * Fresnel: the spectrum C[k] of the sampled 1-D chirp (impulse response of Eq.(3)/(6), P:L113,
//     P:L132, taps d = -N..N-1 stored wrapped at d mod 2N), by a two-step fp64 FFT (sqrt(M) shared-memory
//     transforms per step).  FFT2[h_F](k,l) = Cx[k]*Cy[l] exactly because h_F is separable, so the
//     2N x 2N impulse response and its FFT (the paper's FresnelConvProp + FFT) are never formed.
#include "cwo_internal.h"

namespace cwo {

__global__ void twiddle_kernel(float2* tw, int n) {
    int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= n) return;
    double s, c;
    sincospi(-2.0 * (double)m / (double)n, &s, &c);
    tw[m] = make_float2((float)c, (float)s);
}

__global__ void twiddle64_kernel(double2* tw, int n) {
    int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= n / 2) return;
    double s, c;
    sincospi(-2.0 * (double)m / (double)n, &s, &c);
    tw[m] = make_double2(c, s);
}

cudaError_t build_twiddles(float2* tw, int n, cudaStream_t s) {
    twiddle_kernel<<<(n + 255) / 256, 256, 0, s>>>(tw, n);
    return cudaGetLastError();
}
cudaError_t build_twiddles_f64(double2* tw, int n, cudaStream_t s) {
    twiddle64_kernel<<<(n / 2 + 255) / 256, 256, 0, s>>>(tw, n);
    return cudaGetLastError();
}

__device__ __forceinline__ double2 zmul(double2 a, double2 b) {
    return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}

// Spectrum of the sampled chirp x[n] = exp(i 2 pi a d^2), d = n < M/2 ? n : n - M, a = p0 p1/(2 lambda z) in cycles,
// by a two-step fp64 FFT, M = M1 M2 (n = n1 M2 + n2, k = k1 + M1 k2):
//   step 1 (one CTA per n2 and axis): M1-point transform over n1 in shared memory, times w_M^(n2 k1) -> scratch[k1][n2]
//   step 2 (one CTA per k1 and axis): M2-point transform over n2 -> C[k1 + M1 k2] = coef * X.
// 2 x ~sqrt(M) CTAs of 64 threads instead of one CTA running log2 M global-memory stages (16384 points: 119 -> ~10 us;
// the table build is on the critical path of every propagation with a new z).
constexpr int CHIRP_MAXL = 128;    // M <= 16384 -> M1 <= 128

__device__ __forceinline__ double2 tw_full(const double2* tw64, int idx, int half) {   // w_M^idx, idx < M, table of M/2
    if (idx < half) return tw64[idx];
    const double2 w = tw64[idx - half];
    return make_double2(-w.x, -w.y);
}

// radix-2 Stockham stages of a length-2^l transform held in shared memory (ping-pong a <-> b); returns the buffer
// that holds the result.  w_L^j = w_M^(j M/L).
__device__ double2* smem_fft(double2* a, double2* b, int l, const double2* tw64, int logm) {
    const int L = 1 << l, h = L >> 1;
    for (int lns = 0; lns < l; ++lns) {
        const int ns = 1 << lns;
        for (int j = threadIdx.x; j < h; j += blockDim.x) {
            const int k = j & (ns - 1);
            const double2 w = tw64[(k << (l - 1 - lns)) << (logm - l)];
            const double2 x0 = a[j], x1 = zmul(a[j + h], w);
            const int j0 = ((j >> lns) << (lns + 1)) + k;
            b[j0] = make_double2(x0.x + x1.x, x0.y + x1.y);
            b[j0 + ns] = make_double2(x0.x - x1.x, x0.y - x1.y);
        }
        __syncthreads();
        double2* t = a; a = b; b = t;
    }
    return a;
}

__global__ void __launch_bounds__(64) chirp_step1_kernel(ChirpAxis ax0, ChirpAxis ax1) {
    const ChirpAxis& ax = (blockIdx.y == 0) ? ax0 : ax1;
    const int l1 = (ax.logm + 1) >> 1, l2 = ax.logm - l1, M = 1 << ax.logm, M1 = 1 << l1, M2 = 1 << l2;
    const int n2 = blockIdx.x;
    if (n2 >= M2) return;
    __shared__ double2 buf[2][CHIRP_MAXL];
    for (int n1 = threadIdx.x; n1 < M1; n1 += blockDim.x) {
        const int n = n1 * M2 + n2;
        const double d = (double)((n < M / 2) ? n : n - M);
        double c = ax.a_cycles * d * d;      // |c| <= ~3e3 cycles: fp64 keeps ~1e-13 cycles
        c -= rint(c);
        double s, co;
        sincospi(2.0 * c, &s, &co);
        buf[0][n1] = make_double2(co, s);
    }
    __syncthreads();
    const double2* r = smem_fft(buf[0], buf[1], l1, ax.tw64, ax.logm);
    for (int k1 = threadIdx.x; k1 < M1; k1 += blockDim.x)
        ax.scratch[(size_t)k1 * M2 + n2] = zmul(r[k1], tw_full(ax.tw64, n2 * k1, M / 2));
}

__global__ void __launch_bounds__(64) chirp_step2_kernel(ChirpAxis ax0, ChirpAxis ax1) {
    const ChirpAxis& ax = (blockIdx.y == 0) ? ax0 : ax1;
    const int l1 = (ax.logm + 1) >> 1, l2 = ax.logm - l1, M1 = 1 << l1, M2 = 1 << l2;
    const int k1 = blockIdx.x;
    if (k1 >= M1) return;
    __shared__ double2 buf[2][CHIRP_MAXL];
    for (int n2 = threadIdx.x; n2 < M2; n2 += blockDim.x) buf[0][n2] = ax.scratch[(size_t)k1 * M2 + n2];
    __syncthreads();
    const double2* r = smem_fft(buf[0], buf[1], l2, ax.tw64, ax.logm);
    for (int k2 = threadIdx.x; k2 < M2; k2 += blockDim.x) {
        const int i = k1 + M1 * k2;
        const double2 v = zmul(r[k2], ax.coef);
        if (ax.out) ax.out[i] = make_float2((float)v.x, (float)v.y);
        if (ax.out_pairs) {                                  // planar pairs (even bin, odd bin): lineconv_kernel.cuh
            float* q = reinterpret_cast<float*>(ax.out_pairs + (i >> 1)) + (i & 1);
            q[0] = (float)v.x; q[2] = (float)v.y;
        }
    }
}

cudaError_t build_chirp_spectrum(const ChirpAxis& ax0, const ChirpAxis& ax1, cudaStream_t s) {
    const int lm = ax0.logm > ax1.logm ? ax0.logm : ax1.logm;
    const int l1 = (lm + 1) >> 1;
    chirp_step1_kernel<<<dim3(1 << (lm - l1), 2), 64, 0, s>>>(ax0, ax1);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    chirp_step2_kernel<<<dim3(1 << l1, 2), 64, 0, s>>>(ax0, ax1);
    return cudaGetLastError();
}

// ASM split path (S2): per plane, theta_x[k] = frac(c0 - ax ks^2), theta_y[l] = frac(-ay ls^2) in cycles.
// ax ks^2 reaches ~5e3 cycles (c3, z = 0.5 m): formed in fp64, reduced mod 1, then rounded to fp32.
__global__ void asm_phase_kernel(float* tab, float* resc, const __grid_constant__ AsmPlaneBatch planes, int mx, int my) {
    const AsmPlane pl = planes.p[blockIdx.y];
    if (resc && blockIdx.x == 0 && threadIdx.x == 0) resc[blockIdx.y] = (float)pl.kz;
    float* t = tab + (size_t)blockIdx.y * (mx + my);
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < mx + my; i += gridDim.x * blockDim.x) {
        const bool isx = i < mx;
        const int j = isx ? i : i - mx, m = isx ? mx : my;
        const double b = (double)((j < m / 2) ? j : j - m);
        double c = (isx ? pl.c0 : 0.0) - (isx ? pl.ax : pl.ay) * b * b + (isx ? pl.ox : pl.oy) * b;
        c -= rint(c);
        t[i] = (float)c;
    }
    // Launched with programmatic stream serialization when the table is the plan's own: it depends on nothing earlier
    // in the stream (its previous reader finished before the preceding kernel let this one start), so it is computed
    // while that kernel drains; completing only after it keeps the stream's order for everything that follows.
    asm volatile("griddepcontrol.wait;" ::: "memory");
}

// early: the destination is memory that no kernel still running in the stream can be reading (the plan's own table);
// otherwise (tables inside the caller's workspace, which the previous call's last kernel may still read) the kernel is
// launched as an ordinary, fully ordered one and its griddepcontrol.wait is a no-op.
cudaError_t build_asm_phase_tables(float* tab, float* resc, const AsmPlaneBatch& planes, int n_planes, int mx, int my,
                                   cudaStream_t s, bool early) {
    dim3 grid((mx + my + 255) / 256 > 64 ? 64 : (mx + my + 255) / 256, n_planes);
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = dim3(256); cfg.dynamicSmemBytes = 0; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = early ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, asm_phase_kernel, tab, resc, planes, mx, my);
}

// Quadratic-phase tables of the Fourier-form and shifted Fresnel diffraction (Eq.(8)-(9), Eq.(11)-(12)):
// t[i] = scale (-1)^(alt i) exp(i 2 pi (c0 + c1 m + c2 m^2)), m = i - n/2 (Eq.(4)); the phase is formed and reduced mod 1
// in fp64 (c2 m^2 reaches 1e4 cycles), then rounded once to fp32.
__global__ void quad_phase_kernel(const __grid_constant__ QuadTabBatch b) {
    const QuadTab& t = b.t[blockIdx.y];
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < t.n; i += gridDim.x * blockDim.x) {
        const double m = (double)(i - t.n / 2);
        double c = t.c0 + (t.c1 + t.c2 * m) * m;
        c -= rint(c);
        double sn, cs;
        sincospi(2.0 * c, &sn, &cs);
        const double sc = (t.alt && (i & 1)) ? -t.scale : t.scale;
        t.out[i] = make_float2((float)(sc * cs), (float)(sc * sn));
    }
}

cudaError_t build_quad_phase_tables(const QuadTabBatch& b, int n_tabs, cudaStream_t s) {
    int nmax = 1;
    for (int i = 0; i < n_tabs; ++i) nmax = b.t[i].n > nmax ? b.t[i].n : nmax;
    quad_phase_kernel<<<dim3((nmax + 255) / 256, n_tabs), 256, 0, s>>>(b);
    return cudaGetLastError();
}

}  // namespace cwo
