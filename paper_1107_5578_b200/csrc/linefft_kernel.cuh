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

template <int LOGN>
static cudaError_t launch_linefft_impl(cudaStream_t s, const LineFftParams& p) {
    return p.inverse ? launch_linefft_inst<LOGN, true>(s, p) : launch_linefft_inst<LOGN, false>(s, p);
}

}  // namespace cwo
