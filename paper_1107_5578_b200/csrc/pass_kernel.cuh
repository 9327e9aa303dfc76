// pass_kernel.cuh -- one streaming pass over the field: every CTA loads a tile of W lanes x n points,
// transforms it on chip and stores it.  The three passes of a propagation
// are instances of this kernel:
//   KIND_FWD     load -> FFT -> store                         (row pass R; column pass of the stack)
//   KIND_INV     load -> IFFT -> store                        (row pass R')
//   KIND_FUSED   load -> FFT -> x H -> IFFT -> store          (column pass C: S4 second half, S5, S6 first half)
//   KIND_MIDINV  load -> x H -> IFFT -> store                 (stack: column pass per plane, S9)
// Zero padding (S3) and cropping (S8) are point-validity bounds of the load / store; the GS
// constraints (S10) are load/store modes; H (S2) is produced in registers by mid().
#pragma once
#include "cwo_internal.h"
#include "fft_core.cuh"

namespace cwo {

__device__ __forceinline__ size_t addr_of(const Addr& a, long long tile_off, int w, int p) {
    return (size_t)tile_off + (size_t)w * a.lane_stride + (size_t)(p >> a.sh) * a.hi_stride +
           (size_t)(p & a.mask) * a.lo_stride;
}

// Transfer-function multiply for one unit: register e holds point l = u + e*Q of lane k.
// Computes v <- conj(v * m) so that the following forward transform acts as the inverse one.
template <int LOGN>
__device__ __forceinline__ void mid_unit(float2 (&v)[16], int u, int lane, const PassParams& P) {
    constexpr int N = 1 << LOGN, Q = N / 16;
    if (P.mid_mode == MID_TABLES) {
        // Fresnel: FFT2 of the sampled separable chirp is the outer product Cx[k]*Cy[l]
        float2 cx = __ldg(&P.tab_lane[lane]);
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            float2 m = cmul(cx, __ldg(&P.tab_point[u + e * Q]));
            v[e] = cconj(cmul(v[e], m));
        }
    } else if (P.mid_mode == MID_ASM_F64) {
        // Eq.(16) P:L203 with the phase in cycles evaluated in fp64:
        // w = 1/lambda^2 - (fx^2 + fy^2) (same expression and rounding as the oracle's evanescent test)
        int ks = (lane < P.n_lane_bins / 2) ? lane : lane - P.n_lane_bins;
        double fx = (double)ks * P.df_lane;
        double fx2 = __dmul_rn(fx, fx);
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            int l = u + e * Q;
            int ls = (l < N / 2) ? l : l - N;
            double fy = (double)ls * P.df_point;
            double w = __dsub_rn(P.inv_lam2, __dadd_rn(fx2, __dmul_rn(fy, fy)));
            float2 m = make_float2(0.f, 0.f);
            if (w >= 0.0) {
                double c = P.z * sqrt(w);
                c -= rint(c);
                float s, co;
                sincospif(2.0f * (float)c, &s, &co);
                m = make_float2(co * P.mid_scale, s * P.mid_scale);
            }
            v[e] = cconj(cmul(v[e], m));
        }
    } else if (P.mid_mode == MID_ASM_SPLIT) {
        // H = c0*Ex[k] * Ey[l] * exp(-i 2 pi res), res = (z/lambda) s^2 / (2 (1+sqrt(1-s))^2),
        // s = lambda^2 (fx^2 + fy^2): constant and paraxial parts from fp64 1-D tables, the small
        // non-paraxial residual in fp32 (no cancellation).  Only used when no bin is evanescent.
        int ks = (lane < P.n_lane_bins / 2) ? lane : lane - P.n_lane_bins;
        float2 ex = __ldg(&P.tab_lane[lane]);
        float sx = P.res_a * (float)ks * (float)ks;          // lambda^2 fx^2
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            int l = u + e * Q;
            int ls = (l < N / 2) ? l : l - N;
            float s = fmaf(P.res_b * (float)ls, (float)ls, sx);
            float r = 1.0f + sqrtf(1.0f - s);
            float res = P.res_c * s * s / (2.0f * r * r);       // cycles
            res -= rintf(res);
            float sn, cs;
            sincospif(-2.0f * res, &sn, &cs);
            float2 m = cmul(cmul(ex, __ldg(&P.tab_point[l])), make_float2(cs, sn));
            v[e] = cconj(cmul(v[e], m));
        }
    }
}

template <int LOGN, int KIND>
__global__ void __launch_bounds__(tile_threads(LOGN), tile_minblocks(LOGN))
pass_kernel(const __grid_constant__ PassParams P) {
    constexpr int LOGW = tile_logw(LOGN), W = 1 << LOGW, T = tile_threads(LOGN), UPT = tile_upt(LOGN);
    constexpr int N = 1 << LOGN, Q = N / 16;
    extern __shared__ float2 sm[];

    const int tile = blockIdx.x;
    int uu[UPT], ww[UPT];
    bool ok[UPT];
#pragma unroll
    for (int it = 0; it < UPT; ++it) {
        int unit = threadIdx.x + it * T;
        ww[it] = unit & (W - 1);
        uu[it] = unit >> LOGW;
        ok[it] = (tile * W + ww[it]) < P.lanes_total;
    }

    float2 v[UPT][16];
    // ---- load (zero padding = points >= p_in_valid) ------------------------------------------
    {
        const long long toff = (long long)tile * P.ain.tile_stride;
#pragma unroll
        for (int it = 0; it < UPT; ++it) {
#pragma unroll
            for (int e = 0; e < 16; ++e) {
                int p = uu[it] + e * Q;
                float2 x = make_float2(0.f, 0.f);
                if (ok[it] && p < P.p_in_valid) {
                    if (P.in_mode == IN_COMPLEX) {
                        x = P.in[addr_of(P.ain, toff, ww[it], p)];
                    } else {   // GS step 1: amp * exp(i phase)  (Listing 8 lines 3-5)
                        size_t a = (size_t)(tile * W + ww[it]) * P.aux_pitch + p;
                        float s, c;
                        sincosf(P.in_phase[a], &s, &c);
                        float am = P.in_amp[a];
                        x = make_float2(am * c, am * s);
                    }
                }
                if constexpr (KIND == KIND_INV) x = cconj(x);
                v[it][e] = x;
            }
        }
    }

    // ---- transform ---------------------------------------------------------------------------
    if constexpr (KIND == KIND_FWD) {
        fft_tile<LOGN, LOGW, UPT, true>(v, uu, ww, sm, P.tw);
    } else if constexpr (KIND == KIND_INV) {
        fft_tile<LOGN, LOGW, UPT, false>(v, uu, ww, sm, P.tw);
    } else {
        if constexpr (KIND == KIND_FUSED) fft_tile<LOGN, LOGW, UPT, true>(v, uu, ww, sm, P.tw);
#pragma unroll
        for (int it = 0; it < UPT; ++it) mid_unit<LOGN>(v[it], uu[it], tile * W + ww[it], P);
        fft_tile<LOGN, LOGW, UPT, false>(v, uu, ww, sm, P.tw);
    }

    // ---- store (crop = points >= p_out_valid; conj completes the inverse transform) ----------
    {
        const long long toff = (long long)tile * P.aout.tile_stride;
        const float sc = P.out_scale;
#pragma unroll
        for (int it = 0; it < UPT; ++it) {
#pragma unroll
            for (int e = 0; e < 16; ++e) {
                int p = uu[it] + e * Q;
                if (!(ok[it] && p < P.p_out_valid)) continue;
                float2 x = v[it][e];
                if constexpr (KIND != KIND_FWD) x.y = -x.y;
                if (P.out_mode == OUT_COMPLEX) {
                    P.out[addr_of(P.aout, toff, ww[it], p)] = make_float2(x.x * sc, x.y * sc);
                } else {
                    size_t a = (size_t)(tile * W + ww[it]) * P.aux_pitch + p;
                    if (P.out_mode == OUT_PHASOR_AMP) {
                        // phase constraint then amplitude constraint (Listing 8 lines 11-13 / 15-16):
                        // keep u/|u| (1 where u == 0), replace the amplitude by that of the next plane
                        float m2 = x.x * x.x + x.y * x.y;
                        float am = P.out_amp[a];
                        float2 ph = make_float2(1.f, 0.f);
                        if (m2 > 0.f) { float r = rsqrtf(m2); ph = make_float2(x.x * r, x.y * r); }
                        P.out[addr_of(P.aout, toff, ww[it], p)] = make_float2(am * ph.x, am * ph.y);
                    } else {   // OUT_PHASE: Eq.(25) P:L482 as atan2
                        reinterpret_cast<float*>(P.out)[a] = atan2f(x.y, x.x);
                    }
                }
            }
        }
    }
}

template <int LOGN, int KIND>
static cudaError_t launch_one(int n_tiles, cudaStream_t s, const PassParams& p) {
    constexpr size_t smem = TileShape<LOGN, tile_logw(LOGN)>::SMEM_BYTES;
    static bool configured = false;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(pass_kernel<LOGN, KIND>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)smem);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    pass_kernel<LOGN, KIND><<<n_tiles, tile_threads(LOGN), smem, s>>>(p);
    return cudaGetLastError();
}

template <int LOGN>
static cudaError_t launch_pass_impl(int kind, int n_tiles, cudaStream_t s, const PassParams& p) {
    switch (kind) {
        case KIND_FWD: return launch_one<LOGN, KIND_FWD>(n_tiles, s, p);
        case KIND_INV: return launch_one<LOGN, KIND_INV>(n_tiles, s, p);
        case KIND_FUSED: return launch_one<LOGN, KIND_FUSED>(n_tiles, s, p);
        case KIND_MIDINV: return launch_one<LOGN, KIND_MIDINV>(n_tiles, s, p);
    }
    return cudaErrorInvalidValue;
}

}  // namespace cwo
