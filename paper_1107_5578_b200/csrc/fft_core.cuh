// fft_core.cuh -- register/shared-memory FFT building blocks (complex64, sm_100a).
//
// A CTA owns a tile of W independent length-n transforms ("lanes", n = 2^LOGN).  The work is cut
// into units of 16 points: unit (u, w), u in [0, n/16), always holds the points u + e*(n/16),
// e = 0..15, of lane w in registers.  A Stockham autosort stage of radix R (2,4,8,16) does 16/R
// butterflies per unit on those registers, then the tile is exchanged through shared memory
// ([point][lane], one pad row every 16 points => conflict-free 64-bit accesses for every stage).
// n = R0 * 16^m with R0 in {1,2,4,8}: the small radix runs first (SMALL_FIRST) or last, so that
// a forward transform ending in a radix-16 stage and an inverse one starting with a radix-16 stage
// hold the same 16 points per unit and can be chained without an exchange (fused column pass).
// Only the forward kernel exp(-i 2 pi jk/n) is implemented; inverse = conj . forward . conj.
//
// Defines the transform of S4/S6 in SURVEY.md section 8(a) (paper: "FFT", "IFFT").
#pragma once
#include <cuda_runtime.h>

namespace cwo {

__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
    return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}
__device__ __forceinline__ float2 csqr(float2 a) {
    return make_float2(fmaf(a.x, a.x, -a.y * a.y), 2.0f * a.x * a.y);
}
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ float2 cconj(float2 a) { return make_float2(a.x, -a.y); }
// a * (-i)
__device__ __forceinline__ float2 cmul_mi(float2 a) { return make_float2(a.y, -a.x); }

#define CWO_C8 0.70710678118654752440f   // cos(pi/4)
#define CWO_C16 0.92387953251128675613f  // cos(pi/8)
#define CWO_S16 0.38268343236508977173f  // sin(pi/8)

// ---- in-register DFTs on v[base + r*S], r = 0..R-1; forward kernel -------------------------
// Output X_q lands at register base + perm<R>(q)*S.
template <int R> __device__ __forceinline__ constexpr int perm(int q) {
    return R == 16 ? ((q & 3) * 4 + (q >> 2)) : R == 8 ? ((q >> 2) + 2 * (q & 3)) : q;
}

template <int S> __device__ __forceinline__ void dft2(float2 (&v)[16], int b) {
    float2 a0 = v[b], a1 = v[b + S];
    v[b] = cadd(a0, a1);
    v[b + S] = csub(a0, a1);
}

// natural-order 4-point DFT on v[b], v[b+S], v[b+2S], v[b+3S]
template <int S> __device__ __forceinline__ void dft4(float2 (&v)[16], int b) {
    float2 a = cadd(v[b], v[b + 2 * S]), c = csub(v[b], v[b + 2 * S]);
    float2 e = cadd(v[b + S], v[b + 3 * S]), d = cmul_mi(csub(v[b + S], v[b + 3 * S]));
    v[b] = cadd(a, e);
    v[b + 2 * S] = csub(a, e);
    v[b + S] = cadd(c, d);
    v[b + 3 * S] = csub(c, d);
}

// 8 = 4 x 2: DFT4 over r2 (inputs r = r1 + 2 r2), twiddle w8^(r1 q2), DFT2 over r1.
template <int S> __device__ __forceinline__ void dft8(float2 (&v)[16], int b) {
    dft4<2 * S>(v, b);
    dft4<2 * S>(v, b + S);
    // r1 = 1: registers b + (1 + 2 q2) S, q2 = 1,2,3
    {
        float2 t = v[b + 3 * S];
        v[b + 3 * S] = make_float2(CWO_C8 * (t.x + t.y), CWO_C8 * (t.y - t.x));   // * (c8, -c8)
        v[b + 5 * S] = cmul_mi(v[b + 5 * S]);
        t = v[b + 7 * S];
        v[b + 7 * S] = make_float2(CWO_C8 * (t.y - t.x), -CWO_C8 * (t.x + t.y));  // * (-c8, -c8)
    }
#pragma unroll
    for (int q2 = 0; q2 < 4; ++q2) dft2<S>(v, b + 2 * q2 * S);
}

// 16 = 4 x 4 (S = 1 only): DFT4 over r2 (r = r1 + 4 r2), twiddle w16^(r1 q2), DFT4 over r1.
__device__ __forceinline__ void dft16(float2 (&v)[16]) {
#pragma unroll
    for (int r1 = 0; r1 < 4; ++r1) dft4<4>(v, r1);
    // v[r1 + 4 q2] *= w16^(r1 q2), w16^m = (cos(pi m/8), -sin(pi m/8))
    v[5] = cmul(v[5], make_float2(CWO_C16, -CWO_S16));     // m = 1
    v[6] = cmul(v[6], make_float2(CWO_C8, -CWO_C8));       // m = 2
    v[7] = cmul(v[7], make_float2(CWO_S16, -CWO_C16));     // m = 3
    v[9] = cmul(v[9], make_float2(CWO_C8, -CWO_C8));       // m = 2
    v[10] = cmul_mi(v[10]);                                // m = 4
    v[11] = cmul(v[11], make_float2(-CWO_C8, -CWO_C8));    // m = 6
    v[13] = cmul(v[13], make_float2(CWO_S16, -CWO_C16));   // m = 3
    v[14] = cmul(v[14], make_float2(-CWO_C8, -CWO_C8));    // m = 6
    v[15] = cmul(v[15], make_float2(-CWO_C16, CWO_S16));   // m = 9
#pragma unroll
    for (int q2 = 0; q2 < 4; ++q2) dft4<1>(v, 4 * q2);
}

template <int R> __device__ __forceinline__ void dftR(float2 (&v)[16], int b) {
    if constexpr (R == 16) dft16(v);
    else if constexpr (R == 8) dft8<2>(v, b);
    else if constexpr (R == 4) dft4<4>(v, b);
    else dft2<8>(v, b);
}

// v[b + r*S] *= w1^r, r = 1..R-1.  Powers by squaring/multiplying (depth <= 4 products).
template <int R> __device__ __forceinline__ void twiddle(float2 (&v)[16], int b, float2 w1) {
    constexpr int S = 16 / R;
    v[b + S] = cmul(v[b + S], w1);
    if constexpr (R >= 4) {
        float2 w2 = csqr(w1), w3 = cmul(w2, w1);
        v[b + 2 * S] = cmul(v[b + 2 * S], w2);
        v[b + 3 * S] = cmul(v[b + 3 * S], w3);
        if constexpr (R >= 8) {
            float2 w4 = csqr(w2), w5 = cmul(w4, w1), w6 = csqr(w3), w7 = cmul(w4, w3);
            v[b + 4 * S] = cmul(v[b + 4 * S], w4);
            v[b + 5 * S] = cmul(v[b + 5 * S], w5);
            v[b + 6 * S] = cmul(v[b + 6 * S], w6);
            v[b + 7 * S] = cmul(v[b + 7 * S], w7);
            if constexpr (R >= 16) {
                float2 w8 = csqr(w4);
                v[b + 8 * S] = cmul(v[b + 8 * S], w8);
                v[b + 9 * S] = cmul(v[b + 9 * S], cmul(w8, w1));
                v[b + 10 * S] = cmul(v[b + 10 * S], csqr(w5));
                v[b + 11 * S] = cmul(v[b + 11 * S], cmul(w8, w3));
                v[b + 12 * S] = cmul(v[b + 12 * S], csqr(w6));
                v[b + 13 * S] = cmul(v[b + 13 * S], cmul(w8, w5));
                v[b + 14 * S] = cmul(v[b + 14 * S], csqr(w7));
                v[b + 15 * S] = cmul(v[b + 15 * S], cmul(w8, w7));
            }
        }
    }
}

// shared-memory index of (point p, lane w): one pad row of W elements every 16 points
template <int LOGW> __device__ __forceinline__ int sidx(int p, int w) { return ((p + (p >> 4)) << LOGW) + w; }

template <int LOGN, int LOGW> struct TileShape {
    static constexpr int N = 1 << LOGN, W = 1 << LOGW, Q = N / 16;
    static constexpr int SMEM_ELEMS = (N + N / 16) * W;
    static constexpr size_t SMEM_BYTES = sizeof(float2) * (size_t)SMEM_ELEMS;
};

// One Stockham stage (radix 2^LR, Ns = 2^LNS points already combined) on every unit of the thread.
// FIRST: no preceding smem traffic to wait for.  LAST: results stay in registers in natural unit
// order (register e <-> point u + e*Q); otherwise they are exchanged through smem and the thread
// comes back holding the inputs of the next stage.
template <int LOGN, int LOGW, int UPT, int LR, int LNS, bool LAST>
__device__ __forceinline__ void stage(float2 (&v)[UPT][16], const int (&uu)[UPT], const int (&ww)[UPT],
                                      float2* sm, const float2* __restrict__ tw) {
    constexpr int R = 1 << LR, S = 16 / R, Q = (1 << LOGN) / 16, NS = 1 << LNS;
#pragma unroll
    for (int it = 0; it < UPT; ++it) {
#pragma unroll
        for (int i = 0; i < S; ++i) {
            if constexpr (LNS > 0) {
                int j = uu[it] + i * Q;
                int k = j & (NS - 1);
                float2 w1 = __ldg(&tw[k << (LOGN - LNS - LR)]);
                twiddle<R>(v[it], i, w1);
            }
            dftR<R>(v[it], i);
        }
    }
    if constexpr (LAST) {
#pragma unroll
        for (int it = 0; it < UPT; ++it) {
            float2 t[16];
#pragma unroll
            for (int e = 0; e < 16; ++e) t[e] = v[it][e];
#pragma unroll
            for (int i = 0; i < S; ++i)
#pragma unroll
                for (int q = 0; q < R; ++q) v[it][i + q * S] = t[i + perm<R>(q) * S];
        }
    } else {
        __syncthreads();   // everyone has finished reading the previous contents of sm
#pragma unroll
        for (int it = 0; it < UPT; ++it) {
#pragma unroll
            for (int i = 0; i < S; ++i) {
                int j = uu[it] + i * Q;
                int k = j & (NS - 1);
                int j0 = ((j >> LNS) << (LNS + LR)) + k;
#pragma unroll
                for (int q = 0; q < R; ++q)
                    sm[sidx<LOGW>(j0 + (q << LNS), ww[it])] = v[it][i + perm<R>(q) * S];
            }
        }
        __syncthreads();
#pragma unroll
        for (int it = 0; it < UPT; ++it)
#pragma unroll
            for (int e = 0; e < 16; ++e) v[it][e] = sm[sidx<LOGW>(uu[it] + e * Q, ww[it])];
    }
}

// Full forward transform of the tile held in registers (in: register e of unit u = point
// u + e*Q; out: the same mapping in the frequency domain).
template <int LOGN, int LOGW, int UPT, bool SMALL_FIRST>
__device__ __forceinline__ void fft_tile(float2 (&v)[UPT][16], const int (&uu)[UPT], const int (&ww)[UPT],
                                         float2* sm, const float2* __restrict__ tw) {
    constexpr int L0 = LOGN & 3;        // log2 of the small radix (0 = none)
    constexpr int M = LOGN >> 2;        // number of radix-16 stages
    static_assert(M >= 1, "n >= 16");
    if constexpr (SMALL_FIRST) {
        if constexpr (L0 > 0) stage<LOGN, LOGW, UPT, L0, 0, false>(v, uu, ww, sm, tw);
        if constexpr (M >= 1) stage<LOGN, LOGW, UPT, 4, L0, M == 1>(v, uu, ww, sm, tw);
        if constexpr (M >= 2) stage<LOGN, LOGW, UPT, 4, L0 + 4, M == 2>(v, uu, ww, sm, tw);
        if constexpr (M >= 3) stage<LOGN, LOGW, UPT, 4, L0 + 8, M == 3>(v, uu, ww, sm, tw);
    } else {
        if constexpr (M >= 1) stage<LOGN, LOGW, UPT, 4, 0, (M == 1 && L0 == 0)>(v, uu, ww, sm, tw);
        if constexpr (M >= 2) stage<LOGN, LOGW, UPT, 4, 4, (M == 2 && L0 == 0)>(v, uu, ww, sm, tw);
        if constexpr (M >= 3) stage<LOGN, LOGW, UPT, 4, 8, (M == 3 && L0 == 0)>(v, uu, ww, sm, tw);
        if constexpr (L0 > 0) stage<LOGN, LOGW, UPT, L0, 4 * M, true>(v, uu, ww, sm, tw);
    }
}

}  // namespace cwo
