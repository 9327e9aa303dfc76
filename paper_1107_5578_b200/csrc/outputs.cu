// outputs.cu -- the output conversions next to the propagation calls:
//   * Scale, Eq.(21): I256 = (I - min I)/(max I - min I) * 255 -- one min/max reduction, one map;
//   * CGH from point light sources, Eq.(23): I(x,y) = sum_j A_j cos((2 pi/lambda) ((x-x_j)^2 + (y-y_j)^2)/(2 z_j)),
//     an O(N Nx Ny) direct sum bound by the fp32 pipes, not by memory (a different roofline from the FFT passes).
#include <stdint.h>
#include "cwo_internal.h"
#include "fft_packed.cuh"

namespace cwo {

// ---- Scale --------------------------------------------------------------------------------------------------
// order-preserving map float -> uint32 (so that integer atomicMin / atomicMax order floats)
__device__ __forceinline__ unsigned enc_f32(float f) {
    const unsigned u = __float_as_uint(f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float dec_f32(unsigned e) {
    return __uint_as_float((e & 0x80000000u) ? (e & 0x7fffffffu) : ~e);
}

// mm[0] = min (starts at 0xffffffff), mm[1] = max (starts at 0)
__global__ void __launch_bounds__(256) minmax_kernel(const float* __restrict__ in, size_t n, unsigned* mm) {
    unsigned lo = 0xffffffffu, hi = 0u;
    const size_t n4 = n / 4, stride = (size_t)gridDim.x * blockDim.x;
    const float4* in4 = reinterpret_cast<const float4*>(in);
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += stride) {
        const float4 v = __ldcs(&in4[i]);
        const unsigned a = enc_f32(v.x), b = enc_f32(v.y), c = enc_f32(v.z), d = enc_f32(v.w);
        lo = min(min(lo, a), min(b, min(c, d)));
        hi = max(max(hi, a), max(b, max(c, d)));
    }
    for (size_t i = 4 * n4 + (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const unsigned a = enc_f32(in[i]);
        lo = min(lo, a); hi = max(hi, a);
    }
    lo = __reduce_min_sync(0xffffffffu, lo);
    hi = __reduce_max_sync(0xffffffffu, hi);
    __shared__ unsigned slo[8], shi[8];
    if ((threadIdx.x & 31) == 0) { slo[threadIdx.x >> 5] = lo; shi[threadIdx.x >> 5] = hi; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 8; ++w) { lo = min(lo, slo[w]); hi = max(hi, shi[w]); }
        atomicMin(&mm[0], lo); atomicMax(&mm[1], hi);
    }
}

__global__ void __launch_bounds__(256) scale_kernel(const float* __restrict__ in, float* __restrict__ out, size_t n,
                                                    const unsigned* mm) {
    const float lo = dec_f32(mm[0]), hi = dec_f32(mm[1]);
    const float range = hi - lo;
    const size_t n4 = n / 4, stride = (size_t)gridDim.x * blockDim.x;
    const float4* in4 = reinterpret_cast<const float4*>(in);
    float4* out4 = reinterpret_cast<float4*>(out);
    auto f = [&](float v) { return range > 0.f ? (v - lo) / range * 255.0f : 0.0f; };     // constant field -> 0 (R18)
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += stride) {
        const float4 v = __ldcs(&in4[i]);
        __stcs(&out4[i], make_float4(f(v.x), f(v.y), f(v.z), f(v.w)));
    }
    for (size_t i = 4 * n4 + (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) out[i] = f(in[i]);
}

cudaError_t launch_minmax(const float* in, size_t n, unsigned* mm, int n_sm, cudaStream_t s) {
    minmax_kernel<<<n_sm * 8, 256, 0, s>>>(in, n, mm);
    return cudaGetLastError();
}
cudaError_t launch_scale(const float* in, float* out, size_t n, const unsigned* mm, int n_sm, cudaStream_t s) {
    scale_kernel<<<n_sm * 8, 256, 0, s>>>(in, out, n, mm);
    return cudaGetLastError();
}

// ---- point-light-source CGH ---------------------------------------------------------------------------------
// The phase of point j at pixel (x, y) is separable: theta = a_j(x) + b_j(y) with a_j(x) = (x - x_j)^2/(2 lambda z_j)
// cycles (up to ~1e5: formed and reduced mod 1 in fp64), so
//     A cos 2 pi (a + b) = (A cos 2 pi a) cos 2 pi b - (A sin 2 pi a) sin 2 pi b:
// a thread owns C = 4 columns and R = 16 rows; per point it evaluates (A cos, A sin)(a_j(x)) once per column and then
// spends two packed FMAs per column and row PAIR with (cos, sin)(b_j(y)), which the CTA evaluates once per point and
// row and keeps in shared memory as the packed operands.  Per pixel and point: 1/2 FFMA2 x 2, 1/16 LDS.128 (the
// broadcast loads would bound the kernel with one column per thread: 4/C LSU cycles per FMA cycle) and
// (1 fp64 phase + 1 sincos)/R -- no transcendental in the inner loop.
constexpr int PLS_T = 64;      // threads per CTA
constexpr int PLS_C = 4;       // columns per thread (PLS_T apart: coalesced stores)
constexpr int PLS_R = 16;      // rows per CTA
constexpr int PLS_CHUNK = 32;  // points staged per step

// exp(i 2 pi c), c in cycles.  The fraction is taken without conversion instructions (FRND / F2F / MUFU share the 16-lane
// XU pipe, which would bound the kernel): adding 1.5 * 2^20 leaves frac(c) * 2^32 in the low word of the sum (|c| < 2^19),
// an int32 in units of 2^-32 cycles; larger phases (never in the paper's geometry) take the rounding instruction.
__device__ __forceinline__ float2 cis_frac(double c) {
    int q;
    if (fabs(c) < 524288.0) {
        q = __double2loint(c + 1572864.0);
    } else {
        c -= rint(c);
        q = (int)(long long)(c * 4294967296.0);
    }
    float sn, cs;
    __sincosf((float)q * 1.4629180792671596e-9f, &sn, &cs);      // 2 pi / 2^32
    return make_float2(cs, sn);
}

__global__ void __launch_bounds__(PLS_T) pls_cgh_kernel(const double* __restrict__ pts, int npts, float* __restrict__ out,
                                                        int nx, int ny, double px, double py, double lambda) {
    __shared__ ulonglong2 rowcs[PLS_CHUNK][PLS_R / 2];   // (cos b(r), cos b(r+1)), (sin b(r), sin b(r+1)): packed operands
    __shared__ double sx[PLS_CHUNK], sk[PLS_CHUNK];
    __shared__ float sa[PLS_CHUNK];
    const int col0 = blockIdx.x * (PLS_T * PLS_C) + threadIdx.x, row0 = blockIdx.y * PLS_R;
    double x[PLS_C];
#pragma unroll
    for (int c = 0; c < PLS_C; ++c) x[c] = (double)(col0 + c * PLS_T - nx / 2) * px;
    pk acc[PLS_C][PLS_R / 2];
#pragma unroll
    for (int c = 0; c < PLS_C; ++c)
#pragma unroll
        for (int r = 0; r < PLS_R / 2; ++r) acc[c][r] = 0ull;
    for (int j0 = 0; j0 < npts; j0 += PLS_CHUNK) {
        const int m = min(PLS_CHUNK, npts - j0);
        __syncthreads();
        // stage the chunk: per point x_j, 1/(2 lambda z_j), A_j; per point and row the phasor of b_j(y)
        for (int i = threadIdx.x; i < PLS_CHUNK * PLS_R; i += PLS_T) {
            const int jj = i / PLS_R, r = i % PLS_R;
            float2 cs = make_float2(0.f, 0.f);
            if (jj < m) {
                const double* p = pts + 4 * (size_t)(j0 + jj);
                const double k = 1.0 / (2.0 * lambda * p[2]);
                const double dy = (double)(row0 + r - ny / 2) * py - p[1];
                cs = cis_frac(dy * dy * k);
                if (r == 0) { sx[jj] = p[0]; sk[jj] = k; sa[jj] = (float)p[3]; }
            }
            float* q = reinterpret_cast<float*>(&rowcs[jj][r >> 1]);
            q[r & 1] = cs.x; q[2 + (r & 1)] = cs.y;
        }
        __syncthreads();
#pragma unroll 1
        for (int jj = 0; jj < m; ++jj) {
            const double xj = sx[jj], k = sk[jj];
            const float a = sa[jj];
            pk ac[PLS_C], as[PLS_C];
#pragma unroll
            for (int c = 0; c < PLS_C; ++c) {
                const double dx = x[c] - xj;
                const float2 cx = cis_frac(dx * dx * k);
                ac[c] = pk_bcast(a * cx.x); as[c] = pk_bcast(-a * cx.y);
            }
#pragma unroll
            for (int r = 0; r < PLS_R / 2; ++r) {
                const ulonglong2 t = rowcs[jj][r];
#pragma unroll
                for (int c = 0; c < PLS_C; ++c) acc[c][r] = fma2(as[c], t.y, fma2(ac[c], t.x, acc[c][r]));
            }
        }
    }
#pragma unroll
    for (int c = 0; c < PLS_C; ++c) {
        const int col = col0 + c * PLS_T;
        if (col >= nx) continue;
#pragma unroll
        for (int r = 0; r < PLS_R / 2; ++r) {
            float lo, hi;
            pk_split(acc[c][r], lo, hi);
            if (row0 + 2 * r < ny) out[(size_t)(row0 + 2 * r) * nx + col] = lo;
            if (row0 + 2 * r + 1 < ny) out[(size_t)(row0 + 2 * r + 1) * nx + col] = hi;
        }
    }
}

cudaError_t launch_pls_cgh(const double* pts, int npts, float* out, int nx, int ny, double px, double py, double lambda,
                           cudaStream_t s) {
    dim3 grid((nx + PLS_T * PLS_C - 1) / (PLS_T * PLS_C), (ny + PLS_R - 1) / PLS_R);
    pls_cgh_kernel<<<grid, PLS_T, 0, s>>>(pts, npts, out, nx, ny, px, py, lambda);
    return cudaGetLastError();
}

}  // namespace cwo
