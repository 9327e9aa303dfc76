// rowpair_kernel.cuh -- forward row pass (R) over 8192-point rows in packed arithmetic, one CTA per two-row tile.
//
// The persistent row passes of pipe_kernel.cuh need three tile buffers; two 8192-point rows (128 KB) fit once, so this
// length runs one CTA per tile (as pass_kernel.cuh does), but with the even / odd-bin scheme of the pipelined row passes
// instead of scalar butterflies: one radix-2 step (decimation in frequency) turns a row of n = 2h points into two
// h-point lanes with the same twiddles,
//       a[m] = x[m] + x[m+h],  b[m] = (x[m] - x[m+h]) w^m,   X[2j] = FFT_h(a)[j],  X[2j+1] = FFT_h(b)[j],
// i.e. the (slot 0, slot 1) lane pair of fft_packed.cuh, and (X[2j], X[2j+1]) is one planar 16-byte element of the
// column-tiled workspace.  The tile is the four lanes (a, b) of rows 2t, 2t+1; neighbouring threads hold the two rows, so
// every 128-bit store completes a 32-byte sector with its neighbour's.  8192^2 ASM: pass R 348 ->.
#pragma once
#include "pipe_kernel.cuh"

namespace cwo {

template <int LOGN> struct RowPairCfg {
    using CH = Tile<LOGN - 1>;
    static_assert(CH::W == 2, "half-length lanes on lane-pair tiles");
    static constexpr int LOGW = 2;                                   // four lanes: (a, b) of two rows
    static constexpr int T = CH::Q * 2;
    static constexpr size_t EX_BYTES = sizeof(float2) * (size_t)(CH::N + CH::N / 16) * 4;
    static constexpr int NTW = PP<LOGN - 1>::NTW_P;
    static constexpr size_t SMEM = EX_BYTES + 64 + sizeof(float2) * NTW;
};

// PAD (zero-expanded rows, Fresnel / CWO_OPT_ASM_PAD2X): only the first h points are stored, x[m+h] = 0: a = x, b = x w^m
template <int LOGN, bool PAD>
__global__ void __launch_bounds__(RowPairCfg<LOGN>::T, 1) rowpair_fwd_kernel(const __grid_constant__ PassParams P) {
    using K = RowPairCfg<LOGN>;
    using CH = typename K::CH;
    constexpr int QH = CH::Q, H = CH::N;
    extern __shared__ float2 sm[];
    unsigned char* raw = reinterpret_cast<unsigned char*>(sm);
    uint64_t* bars = reinterpret_cast<uint64_t*>(raw + K::EX_BYTES);
    float2* twh = reinterpret_cast<float2*>(raw + K::EX_BYTES + 64);
    if (threadIdx.x == 0) {
        mbar_init(&bars[0], K::T); mbar_init(&bars[1], K::T);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int i = threadIdx.x; i < K::NTW; i += K::T) twh[i] = __ldg(&P.tw[2 * i]);     // h-point twiddles
    const int hus = threadIdx.x >> 1, hr = threadIdx.x & 1;
    const float2 wb = __ldg(&P.tw[hus]);                                                // w^us; w^(us + e QH) = wb w32^e
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const int row = blockIdx.x * 2 + hr;
    // the rows of the CTA that will take this one's place on the SM: have L2 fetch them now (nothing overlaps that
    // CTA's loads: the whole tile goes to registers before the first butterfly)
    if (threadIdx.x < 2 && P.pf_dist > 0 && (int)blockIdx.x + P.pf_dist < P.n_tiles)
        l2_prefetch(P.in + (size_t)((blockIdx.x + P.pf_dist) * 2 + threadIdx.x) * P.pitch, (uint32_t)((PAD ? 1 : 2) * H * sizeof(float2)));
    float2 tq[8];
#pragma unroll
    for (int e = 0; e < 8; ++e) tq[e] = e == 0 ? wb : cmul(wb, w32_pow(e));
    PV pv;
    {
        const float2* x = P.in + (size_t)row * P.pitch + hus;
        float2 lo[16], hi[16];
#pragma unroll
        for (int e = 0; e < 16; ++e) { lo[e] = __ldcs(&x[e * QH]); hi[e] = PAD ? make_float2(0.f, 0.f) : __ldcs(&x[H + e * QH]); }
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            const float2 a = cadd(lo[e], hi[e]), d = csub(lo[e], hi[e]);
            const float2 bb = e < 8 ? cmul(d, tq[e]) : cmul_mi(cmul(d, tq[e - 8]));
            pv.r[e] = pk_make(a.x, bb.x); pv.i[e] = pk_make(a.y, bb.y);
        }
    }
    __syncthreads();
    const SyncSplit sy{&bars[0], &bars[1], 0u, 0u};
    sy.consumed();                                                   // the exchange region starts free
    transform_p<LOGN - 1, true, false, false, MidNone, SyncSplit, K::LOGW>(pv, hus, 2 * hr, sm, twh, MidNone(), sy);
    // [x/2][row][x%2]: the planar pair (2j, 2j+1), j = hus + e QH, of this thread's row
    ulonglong2* out = reinterpret_cast<ulonglong2*>(P.out);
#pragma unroll
    for (int e = 0; e < 16; ++e)
        __stcs(&out[(size_t)(hus + e * QH) * P.ly + row], make_ulonglong2(pv.r[e], pv.i[e]));
}

template <int LOGN, bool PAD>
static cudaError_t launch_rowpair_fwd(int n_tiles, cudaStream_t s, const PassParams& p) {
    using K = RowPairCfg<LOGN>;
    DeviceInfo* d = device_info();
    if (!d) return cudaErrorInvalidDevice;
    static FuncOnce once;
    if (!once.done(d->index)) {
        cudaError_t e = cudaFuncSetAttribute(rowpair_fwd_kernel<LOGN, PAD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)K::SMEM);
        if (e != cudaSuccess) return e;
        once.set(d->index);
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)n_tiles); cfg.blockDim = dim3((unsigned)K::T);
    cfg.dynamicSmemBytes = K::SMEM; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = n_tiles <= 1024 ? 1 : 0;
    cfg.attrs = at; cfg.numAttrs = 1;
    PassParams q = p;
    q.n_tiles = n_tiles;
    q.pf_dist = d->n_sm;
    return cudaLaunchKernelEx(&cfg, rowpair_fwd_kernel<LOGN, PAD>, q);
}

}  // namespace cwo
