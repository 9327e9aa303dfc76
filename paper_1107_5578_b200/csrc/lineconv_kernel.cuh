// lineconv_kernel.cuh -- convolution-form Fresnel diffraction (Eq.(1)-(6), with the 2N expansion of
// P:L235) as SEPARABLE one-dimensional linear convolutions, and the Gerchberg-Saxton chain built from them.
//
// The sampled impulse response h_F(m,n) = exp(i pi ((m px)^2 + (n py)^2)/(lambda z)) is a product hx(m) hy(n), so
// FFT2[h_F] = Cx[k] Cy[l] (reading R10) and the cropped 2-D linear convolution of Eq.(5) is exactly
//        u2 = conv_y( conv_x(u1, hx), hy ):      a linear convolution of every row, then of every column,
// each cropped to the N stored points.  One line is done in ONE residency: zero-padded 2N-point FFT -> x C ->
// inverse 2N-point FFT -> keep N points, so a propagation moves 8 bytes in and 8 bytes out per sample and axis
// instead of the 80 N^2 bytes of the three-pass 2-D form, and transforms 4 N-point lanes per line and axis
// instead of 6 (the padded intermediate spectrum, 2N wide, is never stored and never transformed along y).
//
// The padded transform of a line is two N-point lanes with the SAME twiddles (decimation in frequency / in time):
//       X[2j]   = FFT_N(x)[j]           = E[j]                y[n] = ( S_e[n] + w^-n S_o[n] ),  n < N,
//       X[2j+1] = FFT_N(x w^n)[j]       = O[j],               S_e/o = unnormalised inverse N-point transforms of
//       w = exp(-i 2 pi / 2N)                                  E[j] C[2j] and O[j] C[2j+1]  (1/(2N) folded into C)
// i.e. exactly the lane pair (slot 0, slot 1) of the packed arithmetic of fft_packed.cuh: the zero half costs
// nothing, the discarded half is never formed.  C is stored per axis as planar pairs (re C[2j], re C[2j+1],
// im C[2j], im C[2j+1]), the register format.  The inverse transform is swap . forward . swap (swap = exchange of
// real and imaginary parts, a register renaming): no conjugation, no negation.
//
// Gerchberg-Saxton (Listing 8) alternates P(-z) and P(+z) with a pointwise constraint between them.
// The two 1-D convolutions of a propagation commute, so consecutive propagations are run X Y | Y X | X Y ...:
// the last convolution of one propagation, the constraint (phase kept, amplitude replaced: S10) and the first
// convolution of the next act on the same lines and are fused into one residency (NCONV == 2).  Between passes
// the field is transposed (transpose_kernel) so that every pass reads and writes whole contiguous lines.
#pragma once
#include "pipe_kernel.cuh"
#include "fold_kernel.cuh"     // w32_pow

namespace cwo {

enum ConvIn { CONV_IN_COMPLEX = 0, CONV_IN_AMP_PHASE = 1, CONV_IN_COMPLEX_PRE = 2 };   // _PRE: x pre[n] on load, x post[n] on store
enum ConvOut { CONV_OUT_COMPLEX = 0, CONV_OUT_PHASE = 1 };

// x C, then swap re <-> im (opens the inverse transform)
struct MidConv {
    const ulonglong2* tab; int us, q;
    __device__ __forceinline__ void packed(PV& v) const {
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            const ulonglong2 c = __ldg(&tab[us + e * q]);               // (cr_e, cr_o), (ci_e, ci_o)
            const pk r = v.r[e], i = v.i[e];
            v.i[e] = fma2(r, c.x, pk_neg(mul2(i, c.y)));                 // swapped: new imaginary = real part of the product
            v.r[e] = fma2(r, c.y, mul2(i, c.x));
        }
    }
};

template <int LOGN> struct ConvCfg {
    using C = Tile<LOGN>;
    // One CTA per SM (n = 8192): PERSISTENT CTAs that take tiles from a device counter (first come, first served: static
    // assignment cannot follow the SM-to-SM spread) and prefetch their next tile into shared memory by TMA.
    // Two CTAs per SM (n <= 4096): one CTA per tile; each CTA asks L2 to prefetch the tile of the CTA that will take its
    // place (cp.async.bulk.prefetch.L2), so that tile's first loads find their data on chip.
    static constexpr bool PREFETCH = (C::MINB == 1);
    static constexpr size_t BAR_OFF = C::SMEM_BYTES;
    static constexpr size_t TW_OFF = BAR_OFF + 64;
    static constexpr int NTW = PP<LOGN>::NTW_P;            // stage twiddles, copied to shared memory once per CTA
    static constexpr size_t PF_OFF = (TW_OFF + sizeof(float2) * NTW + 127) / 128 * 128;
    static constexpr size_t PF_BYTES = sizeof(float2) * (size_t)C::N * (C::W / 2);
    static constexpr size_t SMEM = PREFETCH ? PF_OFF + PF_BYTES : PF_OFF;
};

// 8-byte asynchronous copy global -> shared (LSU path; completion by cp.async.wait_group of the issuing thread)
__device__ __forceinline__ void cp_async8(void* dst, const void* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}

// GATHER: the lines are the columns of a row-major field (sample n of line l at in[n * in_stride + l]); the output is
// always written as contiguous lines, i.e. in the transposed layout, which is what the other axis' pass gathers from:
// the two axes alternate without any transpose pass.  The 32-byte sector a sample sits in also holds the samples of
// the three neighbouring lines, which other CTAs request within a microsecond (tiles are handed out in order): HBM
// still moves every sector once, L2 serves it four times.
template <int LOGN, int IN, int NCONV, int OUT, bool GATHER>
__global__ void __launch_bounds__(Tile<LOGN>::T, Tile<LOGN>::MINB) lineconv_kernel(const __grid_constant__ ConvParams P) {
    using C = Tile<LOGN>;
    using K = ConvCfg<LOGN>;
    static_assert(C::PAIR && LOGN >= 8, "lane-pair tiles");
    constexpr int W = C::W, Q = C::Q, N = C::N, H = W / 2;        // H lines per tile
    constexpr bool PF = K::PREFETCH && IN != CONV_IN_AMP_PHASE;
    constexpr bool PREPOST = IN == CONV_IN_COMPLEX_PRE;
    extern __shared__ float2 sm[];
    unsigned char* raw = reinterpret_cast<unsigned char*>(sm);
    uint64_t* bars = reinterpret_cast<uint64_t*>(raw + K::BAR_OFF);      // [0], [1]: SyncSplit; [2]: tile landed
    volatile int* next_tile = reinterpret_cast<volatile int*>(bars + 3);   // persistent form: the CTA's next tile
    float2* tws = reinterpret_cast<float2*>(raw + K::TW_OFF);
    float2* pf = reinterpret_cast<float2*>(raw + K::PF_OFF);
    if (threadIdx.x == 0) {
        mbar_init(&bars[0], C::T); mbar_init(&bars[1], C::T); mbar_init(&bars[2], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int i = threadIdx.x; i < K::NTW; i += C::T) tws[i] = __ldg(&P.tw[i]);
    const float2* tw = tws;
    const int us = threadIdx.x / H, hl = threadIdx.x % H, w0 = 2 * hl;
    const float2 wb = __ldg(&P.tw2[us]);                    // w^us; w^(us + e Q) = wb w32^e
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

    auto fetch = [&](int tile) {                             // thread 0 only
        mbar_expect_tx(&bars[2], (uint32_t)K::PF_BYTES);
        const unsigned char* src = reinterpret_cast<const unsigned char*>(P.in + (size_t)tile * H * N);
        for (uint32_t o = 0; o < K::PF_BYTES; o += 16384u)
            bulk_g2s(reinterpret_cast<unsigned char*>(pf) + o, src + o, 16384u, &bars[2]);
    };
    // gathered prefetch: every thread copies exactly the 16 samples it will read back (its own slots of pf: no barrier)
    auto fetch_gather = [&](int tile) {
        const float2* src = P.in + (size_t)us * P.in_stride + (tile * H + hl);
#pragma unroll
        for (int e = 0; e < 16; ++e) cp_async8(&pf[hl * N + us + e * Q], src + (size_t)e * Q * P.in_stride);
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    if (PF && !GATHER && threadIdx.x == 0) fetch(blockIdx.x);
    if (PF && GATHER) fetch_gather(blockIdx.x);
    if (!K::PREFETCH && !GATHER && threadIdx.x == 0 && (int)blockIdx.x + P.pf_dist < P.n_tiles)
        l2_prefetch(P.in + (size_t)(blockIdx.x + P.pf_dist) * H * N, (uint32_t)K::PF_BYTES);
    // persistent gathered form: tile indices are known one tile ahead (the copies of tile i + 1 start as soon as the
    // registers of tile i are loaded); cur/nxt are uniform over the CTA
    int nxt = 0;
    if (PF && GATHER) {
        if (threadIdx.x == 0) *next_tile = (int)gridDim.x + atomicAdd(P.counter, 1);
    }
    __syncthreads();
    if (PF && GATHER) nxt = *next_tile;

    const SyncSplit sy{&bars[0], &bars[1], 0u, 0u};
    sy.consumed();                                          // the exchange region starts free
    uint32_t it = 0;
#pragma unroll 1
    for (int tile = blockIdx.x; tile < P.n_tiles; ++it) {
        const size_t base = (size_t)(tile * H + hl) * N + us;           // sample n = us + e Q of this thread's line
        // the amplitudes of the constraint are sent for (to L2) a convolution ahead
        if (NCONV > 1 && threadIdx.x == 0) l2_prefetch(P.mid_amp + (size_t)tile * H * N, (uint32_t)(H * N * sizeof(float)));
        // persistent form: the next tile's index is asked for now and used after the first barrier (the round trip of
        // the atomic is covered by the loads)
        int nt = 0;
        if (K::PREFETCH && threadIdx.x == 0) nt = (int)gridDim.x + atomicAdd(P.counter, 1);
        float2 x[16];
        if constexpr (IN == CONV_IN_AMP_PHASE) {
            // GS step 1, Listing 8 lines 3-5: amp exp(i phase) with the accurate sincosf, by a rolled loop staged
            // through the thread's own slots of the (idle) exchange buffer
            __syncthreads();
            float2* mine = sm + threadIdx.x;
#pragma unroll 1
            for (int e = 0; e < 16; ++e) {
                float sn, cs;
                sincosf(P.in_phase[base + e * Q], &sn, &cs);
                const float am = P.in_amp[base + e * Q];
                mine[e * C::T] = make_float2(am * cs, am * sn);
            }
#pragma unroll
            for (int e = 0; e < 16; ++e) x[e] = mine[e * C::T];
            __syncthreads();
        } else if constexpr (PF && GATHER) {
            asm volatile("cp.async.wait_group 0;" ::: "memory");
#pragma unroll
            for (int e = 0; e < 16; ++e) x[e] = pf[hl * N + us + e * Q];
            if (nxt < P.n_tiles) fetch_gather(nxt);          // own slots only: no barrier needed
        } else if constexpr (PF) {
            mbar_wait(&bars[2], it & 1);
#pragma unroll
            for (int e = 0; e < 16; ++e) x[e] = pf[hl * N + us + e * Q];
            __syncthreads();                                 // everybody has its registers: the buffer is free
            if (threadIdx.x == 0) {
                *next_tile = nt;
                if (nt < P.n_tiles) { fence_proxy_async(); fetch(nt); }
            }
        } else if constexpr (GATHER) {
            const float2* src = P.in + (size_t)us * P.in_stride + (tile * H + hl);
#pragma unroll
            for (int e = 0; e < 16; ++e) x[e] = __ldg(src + (size_t)e * Q * P.in_stride);
        } else {
#pragma unroll
            for (int e = 0; e < 16; ++e) x[e] = __ldcs(&P.in[base + e * Q]);   // streamed: keep L1 for the tables
        }
        if constexpr (PREPOST) {                             // Eq.(12): the chirp and ramp factors of the source plane
#pragma unroll
            for (int e = 0; e < 16; ++e) x[e] = cmul(x[e], __ldg(&P.pre[us + e * Q]));
        }

#pragma unroll 1
        for (int c = 0; c < NCONV; ++c) {
            // w^n, n = us + e Q, e < 8;  w^(n + 8Q) = -i w^n
            float2 t[8];
#pragma unroll
            for (int e = 0; e < 8; ++e) t[e] = e == 0 ? wb : cmul(wb, w32_pow(e));
            PV v;                                            // slot 0: x, slot 1: x w^n
#pragma unroll
            for (int e = 0; e < 16; ++e) {
                const float2 m = e < 8 ? cmul(x[e], t[e]) : cmul_mi(cmul(x[e], t[e - 8]));
                v.r[e] = pk_make(x[e].x, m.x); v.i[e] = pk_make(x[e].y, m.y);
            }
            const MidConv mid{P.tab[c], us, Q};
            transform_p<LOGN, true, true, false>(v, us, w0, sm, tw, mid, sy);
            // v = swap(S): S_e + w^-n S_o, with swap(a) conj(w) = swap(a w) ... done on the swapped values:
            // y = S_e + conj(w^n) S_o;  S = (v.i, v.r)
#pragma unroll
            for (int e = 0; e < 8; ++e) t[e] = e == 0 ? wb : cmul(wb, w32_pow(e));
#pragma unroll
            for (int e = 0; e < 16; ++e) {
                float ar, br, ai, bi;
                pk_split(v.i[e], ar, br); pk_split(v.r[e], ai, bi);          // S_e = (ar, ai), S_o = (br, bi)
                float2 wn = e < 8 ? t[e] : cmul_mi(t[e - 8]);
                const float2 m = cmul(make_float2(br, bi), cconj(wn));
                x[e] = make_float2(ar + m.x, ai + m.y);
            }
            if (c + 1 < NCONV) {
                // GS constraints (S10; Listing 8 lines 11-13 / 15-16): keep u/|u| (1 where u == 0), impose the amplitude
                float am[16];
#pragma unroll
                for (int e = 0; e < 16; ++e) am[e] = __ldg(&P.mid_amp[base + e * Q]);
#pragma unroll
                for (int e = 0; e < 16; ++e) {
                    const float m2 = x[e].x * x[e].x + x[e].y * x[e].y;
                    float2 ph = make_float2(1.f, 0.f);
                    if (m2 > 0.f) { const float r = rsqrtf(m2); ph = make_float2(x[e].x * r, x[e].y * r); }
                    x[e] = make_float2(am[e] * ph.x, am[e] * ph.y);
                }
            }
        }

        if constexpr (PREPOST) {                             // Eq.(11): C_S of the destination plane
#pragma unroll
            for (int e = 0; e < 16; ++e) x[e] = cmul(x[e], __ldg(&P.post[us + e * Q]));
        }
        if constexpr (OUT == CONV_OUT_COMPLEX) {
            float2* out = reinterpret_cast<float2*>(P.out);
#pragma unroll
            for (int e = 0; e < 16; ++e) __stcs(&out[base + e * Q], x[e]);
        } else {
            // Eq.(25) P:L482 as atan2, by a rolled loop (atan2f would otherwise be unrolled 16 times)
            __syncthreads();
            float2* mine = sm + threadIdx.x;
#pragma unroll
            for (int e = 0; e < 16; ++e) mine[e * C::T] = x[e];
            float* out = reinterpret_cast<float*>(P.out);
#pragma unroll 1
            for (int e = 0; e < 16; ++e) {
                const float2 y = mine[e * C::T];
                out[base + e * Q] = (y.x == 0.0f && y.y == 0.0f) ? 0.0f : atan2f(y.y, y.x);   // phasor(0) = 1 (cwo.h)
            }
            __syncthreads();
        }
        if constexpr (!K::PREFETCH) break;                   // one CTA per tile
        if constexpr (PF && GATHER) {
            // nt (asked for at the top of this tile) becomes the tile after next
            if (threadIdx.x == 0) *next_tile = nt;
            __syncthreads();
            tile = nxt; nxt = *next_tile;
            __syncthreads();                                 // everybody has read it before thread 0 overwrites it
            continue;
        }
        if constexpr (!PF) { if (threadIdx.x == 0) *next_tile = nt; }
        __syncthreads();
        tile = *next_tile;
    }
    if constexpr (K::PREFETCH) {
        // the counter resets itself: the last CTA to leave zeroes it for the next launch (which reads it only after its
        // griddepcontrol.wait, i.e. after this grid has completed)
        if (threadIdx.x == 0 && atomicAdd(P.counter + 1, 1) == (int)gridDim.x - 1) { P.counter[0] = 0; P.counter[1] = 0; }
    }
}

template <int LOGN, int IN, int NCONV, int OUT, bool GATHER>
static cudaError_t launch_lineconv_gi(cudaStream_t s, const ConvParams& p) {
    using K = ConvCfg<LOGN>;
    DeviceInfo* d = device_info();
    if (!d) return cudaErrorInvalidDevice;
    static FuncOnce once;
    if (!once.done(d->index)) {
        cudaError_t e = cudaFuncSetAttribute(lineconv_kernel<LOGN, IN, NCONV, OUT, GATHER>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, (int)K::SMEM);
        if (e != cudaSuccess) return e;
        once.set(d->index);
    }
    ConvParams q = p;
    q.n_tiles = p.n_lines / (Tile<LOGN>::W / 2);
    const int slots = d->n_sm * Tile<LOGN>::MINB;
    q.pf_dist = slots;
    const int grid = K::PREFETCH ? (q.n_tiles < slots ? q.n_tiles : slots) : q.n_tiles;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3((unsigned)Tile<LOGN>::T);
    cfg.dynamicSmemBytes = K::SMEM; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, lineconv_kernel<LOGN, IN, NCONV, OUT, GATHER>, q);
}
template <int LOGN, int IN, int NCONV, int OUT>
static cudaError_t launch_lineconv_inst(cudaStream_t s, const ConvParams& p) {
    if constexpr (IN != CONV_IN_AMP_PHASE) {
        if (p.gather) return launch_lineconv_gi<LOGN, IN, NCONV, OUT, true>(s, p);
    }
    return launch_lineconv_gi<LOGN, IN, NCONV, OUT, false>(s, p);
}

// variant: 0 plain (complex -> conv -> complex), 1 GS first (amp, phase -> conv -> complex),
//          2 GS middle (complex -> conv, constraint, conv -> complex), 3 GS last (complex -> conv -> phase),
//          4 shifted Fresnel (complex -> x pre -> conv -> x post -> complex)
template <int LOGN>
static cudaError_t launch_lineconv_impl(int variant, cudaStream_t s, const ConvParams& p) {
    switch (variant) {
        case 0: return launch_lineconv_inst<LOGN, CONV_IN_COMPLEX, 1, CONV_OUT_COMPLEX>(s, p);
        case 1: return launch_lineconv_inst<LOGN, CONV_IN_AMP_PHASE, 1, CONV_OUT_COMPLEX>(s, p);
        case 2: return launch_lineconv_inst<LOGN, CONV_IN_COMPLEX, 2, CONV_OUT_COMPLEX>(s, p);
        case 3: return launch_lineconv_inst<LOGN, CONV_IN_COMPLEX, 1, CONV_OUT_PHASE>(s, p);
        case 4: return launch_lineconv_inst<LOGN, CONV_IN_COMPLEX_PRE, 1, CONV_OUT_COMPLEX>(s, p);
    }
    return cudaErrorInvalidValue;
}

}  // namespace cwo
