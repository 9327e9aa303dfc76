// colfold_kernel.cuh -- fused column pass (FFT_y -> x H -> IFFT_y) over 8192-point columns as (even, odd)-bin lane pairs.
//
// pass_kernel.cuh runs this length as two 8192-point lanes: n = 2 * 16^3, so each transform carries a radix-2 stage and
// the fused pair needs 6 exchanges.  One radix-2 step in registers (decimation in frequency going in, in time coming
// out: the scheme of rowpair_kernel.cuh / fold_kernel.cuh / colpad_kernel.cuh) makes a column of n = 2h points the lane pair
//       a[m] = x[m] + x[m+h],  b[m] = (x[m] - x[m+h]) w^m      (X[2j] = FFT_h(a)[j], X[2j+1] = FFT_h(b)[j])
// of the 4096-point transform: 4 exchanges, no radix-2 stage.  The tile is one column pair of the workspace = four
// lanes ((a, b) of columns x, x+1), 512 threads; neighbouring threads hold the two columns of a pair, read the same
// planar 16-byte elements and put their results together by shuffle.  H is applied at the bins (2j, 2j+1) of the slots.
#pragma once
#include "colpad_kernel.cuh"

namespace cwo {

template <int LOGN>
__global__ void __launch_bounds__(ColPadCfg<LOGN>::T, 1) colfold_fused_asm_kernel(const __grid_constant__ PassParams P) {
    using K = ColPadCfg<LOGN>;
    using CH = typename K::CH;
    constexpr int Q = CH::Q, H = CH::N;
    extern __shared__ float2 sm[];
    unsigned char* raw = reinterpret_cast<unsigned char*>(sm);
    uint64_t* bars = reinterpret_cast<uint64_t*>(raw + K::EX_BYTES);
    float2* twh = reinterpret_cast<float2*>(raw + K::EX_BYTES + 64);
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const int tile = blockIdx.x, us = threadIdx.x >> 1, hp = threadIdx.x & 1;
    const float4* src = reinterpret_cast<const float4*>(P.in + (size_t)tile * P.ly * 2);    // [2h rows][16 bytes]
    float4* dst = reinterpret_cast<float4*>(P.out + (size_t)tile * P.ly * 2);
    if (threadIdx.x == 0) {
        if (P.pf_dist > 0 && tile + P.pf_dist < P.n_tiles)
            l2_prefetch(P.in + (size_t)(tile + P.pf_dist) * P.ly * 2, (uint32_t)(P.ly * 16));
        mbar_init(&bars[0], K::T); mbar_init(&bars[1], K::T);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int i = threadIdx.x; i < K::NTW; i += K::T) twh[i] = __ldg(&P.tw[2 * i]);     // h-point twiddles
    const float2 wb = __ldg(&P.tw[us]);                                               // w^us; w^(us + e Q) = wb w32^e
    float2 tq[8];
#pragma unroll
    for (int e = 0; e < 8; ++e) tq[e] = e == 0 ? wb : cmul(wb, w32_pow(e));
    PV pv;                                                            // slot 0: a, slot 1: b  (m = us + e Q)
#pragma unroll
    for (int e = 0; e < 16; ++e) {
        const float4 l4 = __ldcs(&src[us + e * Q]), h4 = __ldcs(&src[H + us + e * Q]);   // both threads of a pair read them
        const float2 lo = hp ? make_float2(l4.y, l4.w) : make_float2(l4.x, l4.z);
        const float2 hi = hp ? make_float2(h4.y, h4.w) : make_float2(h4.x, h4.z);
        const float2 a = cadd(lo, hi), d = csub(lo, hi);
        const float2 bb = e < 8 ? cmul(d, tq[e]) : cmul_mi(cmul(d, tq[e - 8]));
        pv.r[e] = pk_make(a.x, bb.x); pv.i[e] = pk_make(a.y, bb.y);
    }
    const MidAsmPolyEO<LOGN - 1> mid(P, us, 2 * tile + hp);
    __syncthreads();
    const SyncSplit sy{&bars[0], &bars[1], 0u, 0u};
    sy.consumed();                                                   // the exchange region starts free
    transform_p<LOGN - 1, true, true, false, MidAsmPolyEO<LOGN - 1>, SyncSplit, K::LOGW>(pv, us, 2 * hp, sm, twh, mid, sy);
    // conj(y[m]) = S_e' + w^m S_o', conj(y[m+h]) = S_e' - w^m S_o' (S' = the conjugated lane results); the result stays
    // conjugated for pass R'.  Thread hp = 0 writes the elements of rows m, thread hp = 1 those of rows m + h, each with
    // its neighbour's column by shuffle.
#pragma unroll
    for (int e = 0; e < 16; ++e) {
        float ar, br, ai, bi;
        pk_split(pv.r[e], ar, br); pk_split(pv.i[e], ai, bi);
        const float2 t = cmul(make_float2(br, bi), e < 8 ? tq[e] : cmul_mi(tq[e - 8]));
        const float2 ylo = make_float2(ar + t.x, ai + t.y), yhi = make_float2(ar - t.x, ai - t.y);
        const float2 give = hp ? ylo : yhi, keep = hp ? yhi : ylo;
        const float2 got = make_float2(__shfl_xor_sync(0xffffffffu, give.x, 1), __shfl_xor_sync(0xffffffffu, give.y, 1));
        const float2 c0 = hp ? got : keep, c1 = hp ? keep : got;      // columns x, x+1
        __stcs(&dst[hp * H + us + e * Q], make_float4(c0.x, c1.x, c0.y, c1.y));
    }
}

template <int LOGN>
static cudaError_t launch_colfold_fused_asm(int n_tiles, cudaStream_t s, const PassParams& p) {
    using K = ColPadCfg<LOGN>;
    constexpr size_t smem = K::EX_BYTES + 64 + sizeof(float2) * K::NTW;
    DeviceInfo* d = device_info();
    if (!d) return cudaErrorInvalidDevice;
    static FuncOnce once;
    if (!once.done(d->index)) {
        cudaError_t e = cudaFuncSetAttribute(colfold_fused_asm_kernel<LOGN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        once.set(d->index);
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)n_tiles); cfg.blockDim = dim3((unsigned)K::T);
    cfg.dynamicSmemBytes = smem; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = n_tiles <= 1024 ? 1 : 0;
    cfg.attrs = at; cfg.numAttrs = 1;
    PassParams q = p;
    q.n_tiles = n_tiles;
    q.pf_dist = d->n_sm;
    return cudaLaunchKernelEx(&cfg, colfold_fused_asm_kernel<LOGN>, q);
}

}  // namespace cwo
