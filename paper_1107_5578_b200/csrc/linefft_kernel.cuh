// linefft_kernel.cuh -- Fresnel diffraction, Fourier form (Eq.(7)-(9)): ONE transform per axis.
//
//   u2[m2] = c exp(i pi x2^2/(lambda z)) sum_{m1} u1[m1] exp(i pi x1^2/(lambda z)) exp(-+ i 2 pi m1 m2/N),   m = j - N/2,
// per axis (the 2-D form is the product of the two).  With m = j - N/2 the centred kernel is the plain DFT kernel times
// (-1)^(j1 + j2) (N is a multiple of 4), so a line is   out[j2] = post[j2] DFT_N(pre[j1] in[j1])[j2]   with the chirps,
// the alternating signs and (x axis) the coefficient of Eq.(9) in the two fp64-built tables `pre`, `post`
// (tables.cu quad_phase_kernel).  z < 0 flips the sign of the kernel: conj . forward . conj.
// A tile is W whole lines (the lane pairs of fft_packed.cuh = two neighbouring lines); a CTA reads its lines, transforms
// them in registers and writes them back, so the pass may run in place.  The field is transposed between the x pass
// and the y pass (transpose.cu), as in the separable convolution form (lineconv_kernel.cuh).
#pragma once
#include "pipe_kernel.cuh"

namespace cwo {

template <int LOGN, bool INV>
__global__ void __launch_bounds__(Tile<LOGN>::T, Tile<LOGN>::MINB) linefft_kernel(const __grid_constant__ LineFftParams P) {
    using C = Tile<LOGN>;
    static_assert(C::PAIR && LOGN >= 8, "lane-pair tiles");
    constexpr int W = C::W, Q = C::Q, N = C::N, H = W / 2;
    extern __shared__ float2 sm[];
    unsigned char* raw = reinterpret_cast<unsigned char*>(sm);
    uint64_t* bars = reinterpret_cast<uint64_t*>(raw + C::SMEM_BYTES);
    float2* tws = reinterpret_cast<float2*>(raw + C::SMEM_BYTES + 64);
    if (threadIdx.x == 0) {
        mbar_init(&bars[0], C::T); mbar_init(&bars[1], C::T);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int i = threadIdx.x; i < PP<LOGN>::NTW_P; i += C::T) tws[i] = __ldg(&P.tw[i]);
    const int us = threadIdx.x / H, hl = threadIdx.x % H, w0 = 2 * hl;
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    __syncthreads();
    const SyncSplit sy{&bars[0], &bars[1], 0u, 0u};
    sy.consumed();

    // the tile of the CTA that will take this one's place on the SM: have L2 fetch it now (lineconv_kernel.cuh)
    if (threadIdx.x == 0 && P.pf_dist > 0 && (int)blockIdx.x + P.pf_dist < P.n_lines / W)
        l2_prefetch(P.in + (size_t)(blockIdx.x + P.pf_dist) * W * N, (uint32_t)(sizeof(float2) * W * N));
    const size_t base = ((size_t)blockIdx.x * W + w0) * N + us;       // point us + e Q of line (tile W + w0), then + N
    PV v;
#pragma unroll
    for (int e = 0; e < 16; ++e) {
        const float2 pr = __ldg(&P.pre[us + e * Q]);
        float2 a = cmul(__ldcs(&P.in[base + e * Q]), pr), b = cmul(__ldcs(&P.in[base + N + e * Q]), pr);
        if (INV) { a.y = -a.y; b.y = -b.y; }
        v.r[e] = pk_make(a.x, b.x); v.i[e] = pk_make(a.y, b.y);
    }
    transform_p<LOGN, true, false, false>(v, us, w0, sm, tws, MidNone(), sy);
#pragma unroll
    for (int e = 0; e < 16; ++e) {
        const float2 po = __ldg(&P.post[us + e * Q]);
        float ar, br, ai, bi;
        pk_split(v.r[e], ar, br); pk_split(v.i[e], ai, bi);
        if (INV) { ai = -ai; bi = -bi; }
        __stcs(&P.out[base + e * Q], cmul(make_float2(ar, ai), po));
        __stcs(&P.out[base + N + e * Q], cmul(make_float2(br, bi), po));
    }
}

template <int LOGN, bool INV>
static cudaError_t launch_linefft_inst(cudaStream_t s, const LineFftParams& p) {
    constexpr size_t smem = Tile<LOGN>::SMEM_BYTES + 64 + sizeof(float2) * PP<LOGN>::NTW_P;
    DeviceInfo* d = device_info();
    if (!d) return cudaErrorInvalidDevice;
    static FuncOnce once;
    if (!once.done(d->index)) {
        cudaError_t e = cudaFuncSetAttribute(linefft_kernel<LOGN, INV>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        once.set(d->index);
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(p.n_lines / Tile<LOGN>::W)); cfg.blockDim = dim3((unsigned)Tile<LOGN>::T);
    cfg.dynamicSmemBytes = smem; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    LineFftParams q = p;
    q.pf_dist = d->n_sm * Tile<LOGN>::MINB;
    return cudaLaunchKernelEx(&cfg, linefft_kernel<LOGN, INV>, q);
}

// 8192-point lines (n = 2 x 16^3: a radix-2 stage and a third exchange in the plain form): one radix-2 step in
// registers, decimation in frequency, makes a line the (even bins, odd bins) lane pair of the 4096-point transform
// (rowpair_kernel.cuh); the tile is the four lanes of two lines, neighbouring threads hold the two lines, and the bins
// (2j, 2j+1) of a line leave as ONE 16-byte store.  322 -> us per pass at 8192^2.
template <int LOGN, bool INV>
__global__ void __launch_bounds__(Tile<LOGN - 1>::Q * 2, 1) linefft_pair_kernel(const __grid_constant__ LineFftParams P) {
    using CH = Tile<LOGN - 1>;
    static_assert(CH::W == 2 && CH::L0 == 0, "half-length lanes on lane-pair tiles, h = 16^m");
    constexpr int QH = CH::Q, H = CH::N, T = QH * 2, N = 2 * H;
    constexpr size_t EX_BYTES = sizeof(float2) * (size_t)(H + H / 16) * 4;
    extern __shared__ float2 sm[];
    unsigned char* raw = reinterpret_cast<unsigned char*>(sm);
    uint64_t* bars = reinterpret_cast<uint64_t*>(raw + EX_BYTES);
    float2* twh = reinterpret_cast<float2*>(raw + EX_BYTES + 64);
    if (threadIdx.x == 0) {
        mbar_init(&bars[0], T); mbar_init(&bars[1], T);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int i = threadIdx.x; i < PP<LOGN - 1>::NTW_P; i += T) twh[i] = __ldg(&P.tw[2 * i]);     // h-point twiddles
    const int hus = threadIdx.x >> 1, hr = threadIdx.x & 1;
    const float2 wb = __ldg(&P.tw[hus]);                                                        // w^us; w^(us + e QH) = wb w32^e
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const size_t line = (size_t)blockIdx.x * 2 + hr;
    if (threadIdx.x < 2 && P.pf_dist > 0 && (int)blockIdx.x + P.pf_dist < P.n_lines / 2)
        l2_prefetch(P.in + ((size_t)(blockIdx.x + P.pf_dist) * 2 + threadIdx.x) * N, (uint32_t)(sizeof(float2) * N));
    float2 tq[8];
#pragma unroll
    for (int e = 0; e < 8; ++e) tq[e] = e == 0 ? wb : cmul(wb, w32_pow(e));
    PV pv;
    {
        const float2* x = P.in + line * N + hus;
        float2 lo[16], hi[16];
#pragma unroll
        for (int e = 0; e < 16; ++e) { lo[e] = __ldcs(&x[e * QH]); hi[e] = __ldcs(&x[H + e * QH]); }
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            float2 l = cmul(lo[e], __ldg(&P.pre[hus + e * QH])), h = cmul(hi[e], __ldg(&P.pre[H + hus + e * QH]));
            if (INV) { l.y = -l.y; h.y = -h.y; }
            const float2 a = cadd(l, h), d = csub(l, h);
            const float2 bb = e < 8 ? cmul(d, tq[e]) : cmul_mi(cmul(d, tq[e - 8]));
            pv.r[e] = pk_make(a.x, bb.x); pv.i[e] = pk_make(a.y, bb.y);
        }
    }
    __syncthreads();
    const SyncSplit sy{&bars[0], &bars[1], 0u, 0u};
    sy.consumed();
    transform_p<LOGN - 1, true, false, false, MidNone, SyncSplit, 2>(pv, hus, 2 * hr, sm, twh, MidNone(), sy);
    float4* out4 = reinterpret_cast<float4*>(P.out + line * N);
    const float4* post4 = reinterpret_cast<const float4*>(P.post);
#pragma unroll
    for (int e = 0; e < 16; ++e) {                          // bins 2j, 2j+1, j = hus + e QH
        float ar, br, ai, bi;
        pk_split(pv.r[e], ar, br); pk_split(pv.i[e], ai, bi);
        if (INV) { ai = -ai; bi = -bi; }
        const float4 po = __ldg(&post4[hus + e * QH]);
        const float2 y0 = cmul(make_float2(ar, ai), make_float2(po.x, po.y)), y1 = cmul(make_float2(br, bi), make_float2(po.z, po.w));
        __stcs(&out4[hus + e * QH], make_float4(y0.x, y0.y, y1.x, y1.y));
    }
}

template <int LOGN, bool INV>
static cudaError_t launch_linefft_pair_inst(cudaStream_t s, const LineFftParams& p) {
    using CH = Tile<LOGN - 1>;
    constexpr size_t smem = sizeof(float2) * (size_t)(CH::N + CH::N / 16) * 4 + 64 + sizeof(float2) * PP<LOGN - 1>::NTW_P;
    DeviceInfo* d = device_info();
    if (!d) return cudaErrorInvalidDevice;
    static FuncOnce once;
    if (!once.done(d->index)) {
        cudaError_t e = cudaFuncSetAttribute(linefft_pair_kernel<LOGN, INV>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        once.set(d->index);
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(p.n_lines / 2)); cfg.blockDim = dim3((unsigned)(CH::Q * 2));
    cfg.dynamicSmemBytes = smem; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    LineFftParams q = p;
    q.pf_dist = d->n_sm;
    return cudaLaunchKernelEx(&cfg, linefft_pair_kernel<LOGN, INV>, q);
}

template <int LOGN>
static cudaError_t launch_linefft_impl(cudaStream_t s, const LineFftParams& p) {
    if constexpr (LOGN == 13) {
        return p.inverse ? launch_linefft_pair_inst<LOGN, true>(s, p) : launch_linefft_pair_inst<LOGN, false>(s, p);
    }
    return p.inverse ? launch_linefft_inst<LOGN, true>(s, p) : launch_linefft_inst<LOGN, false>(s, p);
}

}  // namespace cwo
