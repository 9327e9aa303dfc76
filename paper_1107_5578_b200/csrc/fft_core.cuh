// fft_core.cuh -- register/shared-memory FFT building blocks (complex64, sm_100a).
//
// A CTA owns a tile of W independent length-n transforms ("lanes", n = 2^LOGN).  The work is cut
// into units of 16 points: unit (u, w), u in [0, n/16), holds the points u + e*(n/16), e = 0..15,
// of lane w in registers.  A thread owns two units ("slots"): the same u in two adjacent lanes
// (PAIR: twiddles are shared and shared-memory accesses are 128-bit), or, when the tile has a
// single lane (n = 16384), units u and u + n/32.
// A Stockham autosort stage of radix R (2,4,8,16) does 16/R butterflies per unit on those registers,
// then the tile is exchanged through shared memory ([point][lane], one pad row every 16 points).
// n = R0 * 16^m with R0 in {1,2,4,8}: the small radix runs first in a forward transform and last in
// an inverse one, so that a forward transform (ending in a radix-16 stage) and the following inverse
// one (starting with a radix-16 stage) hold the same 16 points per unit and chain without an
// exchange (fused column pass).  The radix-16 stages run as ONE runtime loop so the code stays
// small enough for the instruction cache.  Only the forward kernel exp(-i 2 pi jk/n) is
// implemented; inverse = conj . forward . conj.
//
// This is the transform of S4/S6 in SURVEY.md section 8(a) (paper: "FFT", "IFFT").
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

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
__device__ __forceinline__ float2 cmul_mi(float2 a) { return make_float2(a.y, -a.x); }   // a * (-i)

#define CWO_C8 0.70710678118654752440f   // cos(pi/4)
#define CWO_C16 0.92387953251128675613f  // cos(pi/8)
#define CWO_S16 0.38268343236508977173f  // sin(pi/8)

// ---- in-register DFTs on v[b + r*S], r = 0..R-1; forward kernel; X_q lands at b + perm<R>(q)*S ----
template <int R> __host__ __device__ constexpr int perm(int q) {
    return R == 16 ? ((q & 3) * 4 + (q >> 2)) : R == 8 ? ((q >> 2) + 2 * (q & 3)) : q;
}

template <int S> __device__ __forceinline__ void dft2(float2 (&v)[16], int b) {
    float2 a0 = v[b], a1 = v[b + S];
    v[b] = cadd(a0, a1);
    v[b + S] = csub(a0, a1);
}

template <int S> __device__ __forceinline__ void dft4(float2 (&v)[16], int b) {   // natural order
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
    float2 t = v[b + 3 * S];
    v[b + 3 * S] = make_float2(CWO_C8 * (t.x + t.y), CWO_C8 * (t.y - t.x));   // * (c8, -c8)
    v[b + 5 * S] = cmul_mi(v[b + 5 * S]);
    t = v[b + 7 * S];
    v[b + 7 * S] = make_float2(CWO_C8 * (t.y - t.x), -CWO_C8 * (t.x + t.y));  // * (-c8, -c8)
#pragma unroll
    for (int q2 = 0; q2 < 4; ++q2) dft2<S>(v, b + 2 * q2 * S);
}

// 16 = 4 x 4: DFT4 over r2 (r = r1 + 4 r2), twiddle w16^(r1 q2), DFT4 over r1.
__device__ __forceinline__ void dft16(float2 (&v)[16]) {
#pragma unroll
    for (int r1 = 0; r1 < 4; ++r1) dft4<4>(v, r1);
    // v[r1 + 4 q2] *= w16^(r1 q2), w16^m = (cos(pi m/8), -sin(pi m/8))
    v[5] = cmul(v[5], make_float2(CWO_C16, -CWO_S16));     // m = 1
    v[6] = make_float2(CWO_C8 * (v[6].x + v[6].y), CWO_C8 * (v[6].y - v[6].x));     // m = 2
    v[7] = cmul(v[7], make_float2(CWO_S16, -CWO_C16));     // m = 3
    v[9] = make_float2(CWO_C8 * (v[9].x + v[9].y), CWO_C8 * (v[9].y - v[9].x));     // m = 2
    v[10] = cmul_mi(v[10]);                                // m = 4
    v[11] = make_float2(CWO_C8 * (v[11].y - v[11].x), -CWO_C8 * (v[11].x + v[11].y));   // m = 6
    v[13] = cmul(v[13], make_float2(CWO_S16, -CWO_C16));   // m = 3
    v[14] = make_float2(CWO_C8 * (v[14].y - v[14].x), -CWO_C8 * (v[14].x + v[14].y));   // m = 6
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

// Powers w^1 .. w^(R-1) by squaring/multiplying (depth <= 4 products).
template <int R> __device__ __forceinline__ void powers(float2 w1, float2 (&w)[16]) {
    w[1] = w1;
    if constexpr (R >= 4) { w[2] = csqr(w1); w[3] = cmul(w[2], w1); }
    if constexpr (R >= 8) { w[4] = csqr(w[2]); w[5] = cmul(w[4], w1); w[6] = csqr(w[3]); w[7] = cmul(w[4], w[3]); }
    if constexpr (R >= 16) {
        w[8] = csqr(w[4]); w[9] = cmul(w[8], w1); w[10] = csqr(w[5]); w[11] = cmul(w[8], w[3]);
        w[12] = csqr(w[6]); w[13] = cmul(w[8], w[5]); w[14] = csqr(w[7]); w[15] = cmul(w[8], w[7]);
    }
}

// v[b + r*S] *= w[r], r = 1..R-1
template <int R> __device__ __forceinline__ void apply_powers(float2 (&v)[16], int b, const float2 (&w)[16]) {
    constexpr int S = 16 / R;
#pragma unroll
    for (int r = 1; r < R; ++r) v[b + r * S] = cmul(v[b + r * S], w[r]);
}

// register renaming after the last stage of a transform: register i + q*S <- X_q of butterfly i
template <int R> __device__ __forceinline__ void unpermute(float2 (&v)[16]) {
    constexpr int S = 16 / R;
    float2 t[16];
#pragma unroll
    for (int e = 0; e < 16; ++e) t[e] = v[e];
#pragma unroll
    for (int i = 0; i < S; ++i)
#pragma unroll
        for (int q = 0; q < R; ++q) v[i + q * S] = t[i + perm<R>(q) * S];
}

// ---- tile configuration (one place: host sizing and kernels must agree) -----------------------
#ifndef CWO_LOGW12
#define CWO_LOGW12 1
#endif
#ifndef CWO_LOGW13
#define CWO_LOGW13 1
#endif
constexpr int tile_logw(int logn) {
    return logn <= 5 ? 5 : logn <= 9 ? 4 : logn == 10 ? 3 : logn == 11 ? 2 : logn == 12 ? CWO_LOGW12 : logn == 13 ? CWO_LOGW13 : 0;
}
template <int LOGN> struct Tile {
    static constexpr int N = 1 << LOGN, Q = N / 16;
    static constexpr int LOGW = tile_logw(LOGN), W = 1 << LOGW;
    static constexpr bool PAIR = W >= 2;               // a thread's two slots are adjacent lanes
    static constexpr int T = PAIR ? Q * (W / 2) : Q / 2;
#ifndef CWO_MINB
#define CWO_MINB 2
#endif
    static constexpr int MINB = (LOGN <= 13 && T <= 256) ? CWO_MINB : 1;
    static constexpr int L0 = LOGN & 3, M = LOGN >> 2; // n = 2^L0 * 16^M
    static constexpr size_t SMEM_BYTES = sizeof(float2) * (size_t)(N + N / 16) * W;
    // unit-pair variants: one plane per lane, 2 pad elements every 16 points, plane offsets staggered
    // over the banks (16/W elements mod 16)
    static constexpr int XPLANE = N + N / 8 + (W >= 2 ? 16 / W : 8);
    static constexpr size_t SMEM_BYTES_X = sizeof(float2) * (size_t)W * (size_t)XPLANE;
};

// ---- mbarrier primitives (shared::cta) ------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* b, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* b, uint32_t parity) {
    uint32_t ok;
    do {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(ok)
            : "r"(smem_u32(b)), "r"(parity)
            : "memory");
    } while (!ok);
}
__device__ __forceinline__ void mbar_arrive(uint64_t* b) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}

__device__ __forceinline__ void mbar_expect_tx(uint64_t* b, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
// global -> shared bulk copy (TMA, no tensor map), completion counted in bytes on the mbarrier
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
// ask L2 to fetch a contiguous block (multiple of 16 bytes); no destination, no completion
__device__ __forceinline__ void l2_prefetch(const void* src, uint32_t bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
}
// order this thread's generic-proxy accesses to shared memory before later async-proxy (bulk copy) writes
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// Barrier over the threads that share a tile: the whole CTA (one tile per CTA), or a named barrier over
// one 256-thread group of a persistent CTA that keeps several tiles in flight (pipe_kernel.cuh).
// An exchange between two stages needs two synchronisations: war() before the stores (everybody has loaded
// the previous contents of the region; a thread announces that with consumed() right after its loads) and
// raw() before the loads (everybody's stores are visible; raw_arrive() ... raw_wait() when there is work that
// needs neither, such as the next stage's twiddle powers).  With plain barriers consumed() and raw_arrive() are empty.
struct SyncCta {
    static constexpr bool EARLY_WAR = false;   // a blocking barrier belongs right before the stores
    __device__ __forceinline__ void operator()() const { __syncthreads(); }
    __device__ __forceinline__ void consumed() const {}
    __device__ __forceinline__ void war() const { __syncthreads(); }
    __device__ __forceinline__ void raw() const { __syncthreads(); }
    __device__ __forceinline__ void raw_arrive() const {}
    __device__ __forceinline__ void raw_wait() const { __syncthreads(); }
};
struct SyncGroup {
    static constexpr bool EARLY_WAR = false;
    int id;
    __device__ __forceinline__ void operator()() const { asm volatile("bar.sync %0, 256;" ::"r"(id) : "memory"); }
    __device__ __forceinline__ void consumed() const {}
    __device__ __forceinline__ void war() const { (*this)(); }
    __device__ __forceinline__ void raw() const { (*this)(); }
    __device__ __forceinline__ void raw_arrive() const {}
    __device__ __forceinline__ void raw_wait() const { (*this)(); }
};
// Split-phase form on two mbarriers (arrival count = threads of the tile): consumed() arrives on the first one
// a whole butterfly block before war() waits on it, so that wait is normally already satisfied and the stores
// can be issued among the last butterflies.  Both barriers are used once per exchange; n counts the uses.
struct SyncSplit {
    static constexpr bool EARLY_WAR = true;    // the wait is normally satisfied: take it before the butterflies
    uint64_t* bc; uint64_t* bp; mutable uint32_t nc, np;
    __device__ __forceinline__ void operator()() const { __syncthreads(); }
    __device__ __forceinline__ void consumed() const { mbar_arrive(bc); }
    __device__ __forceinline__ void war() const { mbar_wait(bc, nc & 1); ++nc; }
    __device__ __forceinline__ void raw() const { raw_arrive(); raw_wait(); }
    __device__ __forceinline__ void raw_arrive() const { mbar_arrive(bp); }
    __device__ __forceinline__ void raw_wait() const { mbar_wait(bp, np & 1); ++np; }
};

// shared-memory index of (point p, lane w): one pad row of W elements every 16 points
template <int LOGW> __device__ __forceinline__ int sidx(int p, int w) { return ((p + (p >> 4)) << LOGW) + w; }

// Write the outputs of a radix-2^LR stage with Ns = 2^lns to shared memory in Stockham order and read
// back the inputs of the next stage.  u[], w0: the thread's units (see top of file).
template <int LOGN, int LR, class SY>
__device__ __forceinline__ void exchange(float2 (&v)[2][16], const int (&u)[2], int w0, int lns, float2* sm,
                                         const SY& sync) {
    using C = Tile<LOGN>;
    constexpr int R = 1 << LR, S = 16 / R;
    sync();                       // everyone has finished reading the previous contents
    if constexpr (C::PAIR) {
#pragma unroll
        for (int i = 0; i < S; ++i) {
            const int j = u[0] + i * C::Q;
            const int j0 = ((j >> lns) << (lns + LR)) + (j & ((1 << lns) - 1));
#pragma unroll
            for (int q = 0; q < R; ++q) {
                const float2 a = v[0][i + perm<R>(q) * S], b = v[1][i + perm<R>(q) * S];
                *reinterpret_cast<float4*>(&sm[sidx<C::LOGW>(j0 + (q << lns), w0)]) = make_float4(a.x, a.y, b.x, b.y);
            }
        }
        sync();
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            const float4 t = *reinterpret_cast<const float4*>(&sm[sidx<C::LOGW>(u[0] + e * C::Q, w0)]);
            v[0][e] = make_float2(t.x, t.y);
            v[1][e] = make_float2(t.z, t.w);
        }
    } else {
#pragma unroll
        for (int s = 0; s < 2; ++s)
#pragma unroll
            for (int i = 0; i < S; ++i) {
                const int j = u[s] + i * C::Q;
                const int j0 = ((j >> lns) << (lns + LR)) + (j & ((1 << lns) - 1));
#pragma unroll
                for (int q = 0; q < R; ++q) sm[sidx<0>(j0 + (q << lns), 0)] = v[s][i + perm<R>(q) * S];
            }
        sync();
#pragma unroll
        for (int s = 0; s < 2; ++s)
#pragma unroll
            for (int e = 0; e < 16; ++e) v[s][e] = sm[sidx<0>(u[s] + e * C::Q, 0)];
    }
}

// Twiddle (if lns > 0) and butterflies of one radix-2^LR stage on both slots.
template <int LOGN, int LR, bool SEP = !Tile<LOGN>::PAIR, bool TW_SHARED = false>
__device__ __forceinline__ void butterflies(float2 (&v)[2][16], const int (&u)[2], int lns,
                                            const float2* __restrict__ tw) {
    using C = Tile<LOGN>;
    constexpr int R = 1 << LR, S = 16 / R;
#pragma unroll
    for (int i = 0; i < S; ++i) {
        if (lns > 0) {
            float2 w[16];
            const int k0 = (u[0] + i * C::Q) & ((1 << lns) - 1);
            powers<R>(TW_SHARED ? tw[k0 << (LOGN - lns - LR)] : __ldg(&tw[k0 << (LOGN - lns - LR)]), w);
            apply_powers<R>(v[0], i, w);
            if constexpr (SEP) {                  // the two slots are different units: own twiddles
                const int k1 = (u[1] + i * C::Q) & ((1 << lns) - 1);
                powers<R>(TW_SHARED ? tw[k1 << (LOGN - lns - LR)] : __ldg(&tw[k1 << (LOGN - lns - LR)]), w);
            }
            apply_powers<R>(v[1], i, w);
        }
        dftR<R>(v[0], i);
        dftR<R>(v[1], i);
    }
}

// Forward and/or inverse transform of the tile held in registers, with `mid` applied between them
// (mid must also conjugate so that the second forward transform acts as an inverse one).
// In / out: register e of unit u <-> point u + e*Q.
template <int LOGN, bool HAS_FWD, bool HAS_INV, class Mid, class SY>
__device__ __forceinline__ void transform(float2 (&v)[2][16], const int (&u)[2], int w0, float2* sm,
                                          const float2* __restrict__ tw, Mid mid, const SY& sync) {
    using C = Tile<LOGN>;
    constexpr int L0 = C::L0, M = C::M;
    static_assert(M >= 1, "n >= 16");
    if constexpr (HAS_FWD && L0 > 0) {                      // small radix first, no twiddles
        butterflies<LOGN, L0>(v, u, 0, tw);
        exchange<LOGN, L0>(v, u, w0, 0, sm, sync);
    }
    constexpr int NST = (HAS_FWD ? M : 0) + (HAS_INV ? M : 0);
#pragma unroll 1
    for (int s = 0; s < NST; ++s) {
        const bool inv_half = HAS_FWD ? (s >= M) : true;
        const int sl = (HAS_FWD && inv_half) ? s - M : s;
        const int lns = inv_half ? 4 * sl : L0 + 4 * sl;
        butterflies<LOGN, 4>(v, u, lns, tw);
        if (sl == M - 1) {
            if (!inv_half) {                                 // end of the forward transform
                unpermute<16>(v[0]); unpermute<16>(v[1]);
                if constexpr (HAS_INV) mid(v);
                continue;
            }
            if (L0 == 0) { unpermute<16>(v[0]); unpermute<16>(v[1]); break; }
        }
        exchange<LOGN, 4>(v, u, w0, lns, sm, sync);
    }
    if constexpr (!HAS_FWD && HAS_INV) { /* mid (if any) was applied by the caller before the call */ }
    if constexpr (HAS_INV && L0 > 0) {                      // small radix last
        butterflies<LOGN, L0>(v, u, 4 * M, tw);
        unpermute<(1 << L0)>(v[0]); unpermute<(1 << L0)>(v[1]);
    }
}

// ---- unit-pair mapping ---------------------------------------------------------------------------------
// Where a row pass meets the column-tiled workspace T[x/Wc][y][x%Wc], the 16 bytes that are contiguous in
// memory are two neighbouring points (x, x+1) of ONE row.  For that one stage a thread therefore holds
// the units 2i and 2i+1 of lane w (thread = i*W + w) instead of unit u in two adjacent lanes, so that
// global accesses are 128-bit and neighbouring threads cover full 32-byte sectors.

// Forward transform; the LAST stage runs in unit-pair mapping.  In: standard mapping.
// Out: register e of slot s <-> point 2i + s + e*Q of lane w, (w, i) = (t % W, t / W).
template <int LOGN, class SY>
__device__ __forceinline__ void transform_fwd_xlast(float2 (&v)[2][16], int t, float2* sm,
                                                    const float2* __restrict__ tw, const SY& sync) {
    using C = Tile<LOGN>;
    constexpr int L0 = C::L0, M = C::M, Q = C::Q, W = C::W;
    static_assert(C::PAIR && M >= 2, "unit-pair mapping needs a tile of >= 2 lanes");
    const int us = t / (W / 2), w0 = 2 * (t % (W / 2));
    const int u[2] = {us, us};
    if constexpr (L0 > 0) {
        butterflies<LOGN, L0>(v, u, 0, tw);
        exchange<LOGN, L0>(v, u, w0, 0, sm, sync);
    }
#pragma unroll 1
    for (int s = 0; s < M - 2; ++s) {
        butterflies<LOGN, 4>(v, u, L0 + 4 * s, tw);
        exchange<LOGN, 4>(v, u, w0, L0 + 4 * s, sm, sync);
    }
    constexpr int lns = L0 + 4 * (M - 2);
    butterflies<LOGN, 4>(v, u, lns, tw);
    // exchange into one plane per lane, then read back unit pairs
    sync();
    {
        const int j0 = ((us >> lns) << (lns + 4)) + (us & ((1 << lns) - 1));
        float2* pl = sm + w0 * C::XPLANE;
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            const int p = j0 + (q << lns), pi = p + 2 * (p >> 4);
            pl[pi] = v[0][perm<16>(q)];
            pl[C::XPLANE + pi] = v[1][perm<16>(q)];
        }
    }
    sync();
    const int w = t % W, i2 = 2 * (t / W);                 // units i2, i2 + 1 of lane w
#pragma unroll
    for (int e = 0; e < 16; ++e) {
        const int p = i2 + e * Q;
        const float4 x = *reinterpret_cast<const float4*>(&sm[w * C::XPLANE + p + 2 * (p >> 4)]);
        v[0][e] = make_float2(x.x, x.y);
        v[1][e] = make_float2(x.z, x.w);
    }
    const int ux[2] = {i2, i2 + 1};
    butterflies<LOGN, 4, true>(v, ux, L0 + 4 * (M - 1), tw);
    unpermute<16>(v[0]); unpermute<16>(v[1]);
}

// Inverse transform (as conj . forward . conj, the conj being the caller's); the FIRST stage runs in
// unit-pair mapping.  In: register e of slot s <-> point 2i + s + e*Q of lane w.  Out: standard mapping.
template <int LOGN, class SY>
__device__ __forceinline__ void transform_inv_xfirst(float2 (&v)[2][16], int t, float2* sm,
                                                     const float2* __restrict__ tw, const SY& sync) {
    using C = Tile<LOGN>;
    constexpr int L0 = C::L0, M = C::M, Q = C::Q, W = C::W;
    static_assert(C::PAIR && M >= 2, "unit-pair mapping needs a tile of >= 2 lanes");
    const int w = t % W, i2 = 2 * (t / W);
    dft16(v[0]); dft16(v[1]);                               // Ns = 1: no twiddles
    sync();
#pragma unroll
    for (int s = 0; s < 2; ++s)
#pragma unroll
        for (int q = 0; q < 16; ++q) sm[sidx<C::LOGW>(16 * (i2 + s) + q, w)] = v[s][perm<16>(q)];
    sync();
    const int us = t / (W / 2), w0 = 2 * (t % (W / 2));
#pragma unroll
    for (int e = 0; e < 16; ++e) {
        const float4 x = *reinterpret_cast<const float4*>(&sm[sidx<C::LOGW>(us + e * Q, w0)]);
        v[0][e] = make_float2(x.x, x.y);
        v[1][e] = make_float2(x.z, x.w);
    }
    const int u[2] = {us, us};
#pragma unroll 1
    for (int s = 1; s < M; ++s) {
        butterflies<LOGN, 4>(v, u, 4 * s, tw);
        if (L0 == 0 && s == M - 1) { unpermute<16>(v[0]); unpermute<16>(v[1]); break; }
        exchange<LOGN, 4>(v, u, w0, 4 * s, sm, sync);
    }
    if constexpr (L0 > 0) {
        butterflies<LOGN, L0>(v, u, 4 * M, tw);
        unpermute<(1 << L0)>(v[0]); unpermute<(1 << L0)>(v[1]);
    }
}

}  // namespace cwo
