// colpad_kernel.cuh -- fused column pass of the ZERO-EXPANDED angular spectrum method (CWO_OPT_ASM_PAD2X) with the
// zero half pruned: padded columns as (even bins, odd bins) lane pairs.
//
// A column of the 2N-row calculation area holds N stored samples and N zeros; only N of its 2N outputs are kept.
// With one radix-2 step in each direction (the scheme of lineconv_kernel.cuh) its padded transform is two N-point
// lanes with the same twiddles,
//       X[2j] = FFT_N(x)[j],   X[2j+1] = FFT_N(x w^n)[j],      y[n] = S_e[n] + w^-n S_o[n], n < N,   w = exp(-i 2 pi/2N):
// the zero half costs nothing and the discarded half is never formed -- half the butterflies and 4 exchanges instead
// of 6 compared with running the 2N-point transform on the zeros (pass_kernel.cuh / prefetch_kernel.cuh PAD).
// The tile is one column pair of the workspace = four lanes (E, O of columns x, x+1); neighbouring threads hold the two
// columns of a pair.  H is applied at the bins (2j, 2j+1) of the two slots.
#pragma once
#include "pipe_kernel.cuh"

namespace cwo {

// ASM transfer function for the bins l = 2 (us + e Q) + s of slot s, one column (PipeMidAsmSplit::packed_poly with the
// roles of the packed halves exchanged: the slots differ in the point index, not in the lane).  LOGC: log2 of the lane
// length N; the transform length is 2N.
template <int LOGC> struct MidAsmPolyEO {
    using C = Tile<LOGC>;
    const PassParams& P; int us; float sx, thx;
    __device__ __forceinline__ MidAsmPolyEO(const PassParams& P_, int us_, int lane) : P(P_), us(us_) {
        const int ks = (lane < P.n_lane_bins / 2) ? lane : lane - P.n_lane_bins;
        sx = P.res_a * (float)ks * (float)ks;
        thx = __ldg(reinterpret_cast<const float*>(P.tab_lane) + lane);
    }
    __device__ __forceinline__ void packed(PV& v) const {
        constexpr int Q = C::Q;
        const float2* thy2 = reinterpret_cast<const float2*>(P.tab_point);       // (theta_y[2j], theta_y[2j+1])
        const float l0f = (float)(2 * us);
        const pk sx2 = pk_bcast(sx), thx2 = pk_bcast(thx);
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            const float2 ty = __ldg(&thy2[us + e * Q]);
            const float lsf = l0f + (float)(e < 8 ? 2 * e * Q : 2 * (e - 16) * Q);   // signed bin of l = 2j (exact); 2j+1: +1
            const float lsf1 = lsf + 1.0f;
            const pk sv = add2(sx2, pk_make(P.res_b * lsf * lsf, P.res_b * lsf1 * lsf1));
            pk h = fma2(sv, pk_bcast(33.0f / 2048.0f), pk_bcast(21.0f / 1024.0f));
            h = fma2(sv, h, pk_bcast(7.0f / 256.0f));
            h = fma2(sv, h, pk_bcast(5.0f / 128.0f));
            h = fma2(sv, h, pk_bcast(1.0f / 16.0f));
            h = fma2(sv, h, pk_bcast(0.125f));
            pk res = mul2(mul2(mul2(sv, sv), pk_bcast(P.res_c)), h);
            const pk big = pk_bcast(12582912.0f);                  // 1.5 * 2^23: (x + big) - big = rint(x), |x| < 2^22
            res = sub2(res, sub2(add2(res, big), big));
            const pk ph = mul2(sub2(add2(thx2, pk_make(ty.x, ty.y)), res), pk_bcast(6.283185307179586f));
            float p0, p1, sn0, cs0, sn1, cs1;
            pk_split(ph, p0, p1);
            __sincosf(p0, &sn0, &cs0); __sincosf(p1, &sn1, &cs1);
            // conj(x (cs + i sn)) = (xr cs - xi sn) - i (xr sn + xi cs)
            const pk cs2 = pk_make(cs0, cs1), sn2 = pk_make(sn0, sn1), xr = v.r[e], xi = v.i[e];
            v.r[e] = fma2(xr, cs2, pk_neg(mul2(xi, sn2)));
            v.i[e] = fma2(pk_neg(xr), sn2, pk_neg(mul2(xi, cs2)));
        }
    }
};

// LOGN: log2 of the padded transform length 2N
template <int LOGN> struct ColPadCfg {
    using CH = Tile<LOGN - 1>;
    static constexpr int LOGW = 2;                                   // four lanes: (E, O) of two columns
    static constexpr int T = CH::Q * 2;
    static constexpr int MINB = T <= 256 ? 2 : 1;
    static constexpr size_t EX_BYTES = sizeof(float2) * (size_t)(CH::N + CH::N / 16) * 4;
    static constexpr int NTW = PP<LOGN - 1>::NTW_P;
    static constexpr size_t PF_OFF = (EX_BYTES + 64 + sizeof(float2) * NTW + 127) / 128 * 128;
    static constexpr size_t SMEM = PF_OFF + 16 * (size_t)CH::N;     // + the prefetched column pair (N rows x 16 bytes)
};

template <int LOGN>
__global__ void __launch_bounds__(ColPadCfg<LOGN>::T, ColPadCfg<LOGN>::MINB)
colpad_fused_asm_kernel(const __grid_constant__ PassParams P) {
    using K = ColPadCfg<LOGN>;
    using CH = typename K::CH;
    constexpr int Q = CH::Q;
    extern __shared__ float2 sm[];
    unsigned char* raw = reinterpret_cast<unsigned char*>(sm);
    uint64_t* bars = reinterpret_cast<uint64_t*>(raw + K::EX_BYTES);            // [0], [1]: SyncSplit; [2]: tile landed
    float2* twh = reinterpret_cast<float2*>(raw + K::EX_BYTES + 64);
    const float4* pf = reinterpret_cast<const float4*>(raw + K::PF_OFF);       // the prefetched tile: [N rows][16 bytes]
    const uint32_t bytes = (uint32_t)P.ly * 16;
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const int us = threadIdx.x >> 1, hp = threadIdx.x & 1;
    // persistent: one TMA bulk copy brings the next column pair (ly = N stored rows of planar elements
    // (re_x, re_x+1, im_x, im_x+1)) into the spare buffer while the current one is transformed (prefetch_kernel.cuh)
    auto fetch = [&](int tile) {                             // thread 0 only
        mbar_expect_tx(&bars[2], bytes);
        const unsigned char* src = reinterpret_cast<const unsigned char*>(P.in + (size_t)tile * P.ly * 2);
        for (uint32_t o = 0; o < bytes; o += 16384u)
            bulk_g2s(raw + K::PF_OFF + o, src + o, bytes - o < 16384u ? bytes - o : 16384u, &bars[2]);
    };
    if (threadIdx.x == 0) {
        mbar_init(&bars[0], K::T); mbar_init(&bars[1], K::T); mbar_init(&bars[2], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        fetch(blockIdx.x);
    }
    for (int i = threadIdx.x; i < K::NTW; i += K::T) twh[i] = __ldg(&P.tw[2 * i]);     // N-point twiddles
    const float2 wb = __ldg(&P.tw[us]);                                               // w^us; w^(us + e Q) = wb w32^e
    __syncthreads();
    const SyncSplit sy{&bars[0], &bars[1], 0u, 0u};
    sy.consumed();                                                   // the exchange region starts free
    uint32_t it = 0;
#pragma unroll 1
    for (int tile = blockIdx.x; tile < P.n_tiles; tile += gridDim.x, ++it) {
        float4* dst = reinterpret_cast<float4*>(P.out + (size_t)tile * P.ly * 2);
        float2 tq[8];
#pragma unroll
        for (int e = 0; e < 8; ++e) tq[e] = e == 0 ? wb : cmul(wb, w32_pow(e));
        PV pv;                                                        // slot 0: x, slot 1: x w^n  (n = us + e Q)
        mbar_wait(&bars[2], it & 1);
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            const float4 t4 = pf[us + e * Q];                         // both threads of a column pair read the element
            const float2 x = hp ? make_float2(t4.y, t4.w) : make_float2(t4.x, t4.z);
            const float2 m = e < 8 ? cmul(x, tq[e]) : cmul_mi(cmul(x, tq[e - 8]));
            pv.r[e] = pk_make(x.x, m.x); pv.i[e] = pk_make(x.y, m.y);
        }
        __syncthreads();                                              // everybody has its registers: the buffer is free
        if (threadIdx.x == 0 && tile + (int)gridDim.x < P.n_tiles) { fence_proxy_async(); fetch(tile + gridDim.x); }
        const MidAsmPolyEO<LOGN - 1> mid(P, us, 2 * tile + hp);
        transform_p<LOGN - 1, true, true, false, MidAsmPolyEO<LOGN - 1>, SyncSplit, K::LOGW>(pv, us, 2 * hp, sm, twh, mid, sy);
        // conj(y[n]) = S_e' + w^n S_o' (S' = the conjugated lane results), n = us + e Q < N; the result stays conjugated
        // for pass R'.  Thread hp writes the elements e = 8 hp .. 8 hp + 7 of the pair, its neighbour's column by shuffle.
        float2 y[16];
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            float ar, br, ai, bi;
            pk_split(pv.r[e], ar, br); pk_split(pv.i[e], ai, bi);
            const float2 t = cmul(make_float2(br, bi), e < 8 ? tq[e] : cmul_mi(tq[e - 8]));
            y[e] = make_float2(ar + t.x, ai + t.y);
        }
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            // I keep element k + 8 hp and give away my value of element k + 8 (1 - hp)
            const float2 give = hp ? y[k] : y[k + 8];
            const float2 got = make_float2(__shfl_xor_sync(0xffffffffu, give.x, 1), __shfl_xor_sync(0xffffffffu, give.y, 1));
            const float2 keep = hp ? y[k + 8] : y[k];
            const float2 c0 = hp ? got : keep, c1 = hp ? keep : got;      // columns x, x+1
            __stcs(&dst[us + (k + 8 * hp) * Q], make_float4(c0.x, c1.x, c0.y, c1.y));
        }
    }
}

template <int LOGN>
static cudaError_t launch_colpad_fused_asm(int n_tiles, cudaStream_t s, const PassParams& p) {
    using K = ColPadCfg<LOGN>;
    DeviceInfo* d = device_info();
    if (!d) return cudaErrorInvalidDevice;
    static FuncOnce once;
    if (!once.done(d->index)) {
        cudaError_t e = cudaFuncSetAttribute(colpad_fused_asm_kernel<LOGN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)K::SMEM);
        if (e != cudaSuccess) return e;
        once.set(d->index);
    }
    const int slots = d->n_sm * K::MINB;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(n_tiles < slots ? n_tiles : slots)); cfg.blockDim = dim3((unsigned)K::T);
    cfg.dynamicSmemBytes = K::SMEM; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    PassParams q = p;
    q.n_tiles = n_tiles;
    return cudaLaunchKernelEx(&cfg, colpad_fused_asm_kernel<LOGN>, q);
}

}  // namespace cwo
