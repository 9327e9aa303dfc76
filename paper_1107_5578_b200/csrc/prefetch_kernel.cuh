// prefetch_kernel.cuh -- fused column pass (FFT_y x H x IFFT_y) of the PADDED 8192- and 16384-point transforms
// (Fresnel convolution, GS) as a persistent CTA that prefetches its next tile.
//
// These lengths run one 139 KB tile per SM (pass_kernel.cuh), so nothing hides the global load at the top of a
// tile.  A padded column tile only STORES the non-zero half of its rows in memory: at most 64 KB, which fits
// beside the tile buffer.  One TMA bulk copy brings the next tile into that spare buffer while the current one is
// transformed; a tile then starts by reading registers from shared memory.  Results go straight from registers to
// global memory as before.  Arithmetic, tile/unit mapping and synchronisation are those of pass_kernel.cuh: packed
// f32x2 with split-phase exchanges for lane pairs (8192), scalar for the single lane (16384).
#pragma once
#include "pipe_kernel.cuh"

namespace cwo {

template <int LOGN, int MID>
__global__ void __launch_bounds__(Tile<LOGN>::T, 1) colpref_kernel(const __grid_constant__ PassParams P) {
    using C = Tile<LOGN>;
    constexpr int W = C::W, Q = C::Q, N = C::N, NE = 8;     // padded: points >= N/2 are zero / dropped
    extern __shared__ float2 sm[];
    unsigned char* raw = reinterpret_cast<unsigned char*>(sm);
    uint64_t* bars = reinterpret_cast<uint64_t*>(raw + C::SMEM_BYTES);          // [0], [1]: SyncSplit; [2]: tile landed
    float2* pf = reinterpret_cast<float2*>(raw + C::SMEM_BYTES + 64);           // the prefetched tile, [ly][W]
    const uint32_t bytes = (uint32_t)P.ly * W * 8;
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

    auto fetch = [&](int tile) {                             // thread 0 only
        mbar_expect_tx(&bars[2], bytes);
        const unsigned char* src = reinterpret_cast<const unsigned char*>(P.in + (size_t)tile * P.ly * W);
        for (uint32_t o = 0; o < bytes; o += 16384u)
            bulk_g2s(reinterpret_cast<unsigned char*>(pf) + o, src + o, bytes - o < 16384u ? bytes - o : 16384u, &bars[2]);
    };
    if (threadIdx.x == 0) {
        mbar_init(&bars[0], C::T); mbar_init(&bars[1], C::T); mbar_init(&bars[2], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        fetch(blockIdx.x);
    }
    __syncthreads();

    int u[2], w0;
    if constexpr (C::PAIR) {
        w0 = 2 * (threadIdx.x % (W / 2));
        u[0] = u[1] = threadIdx.x / (W / 2);
    } else {
        w0 = 0;
        u[0] = threadIdx.x; u[1] = threadIdx.x + Q / 2;
    }
    const SyncSplit sy{&bars[0], &bars[1], 0u, 0u};
    if constexpr (C::PAIR) sy.consumed();                    // the exchange region starts free

    uint32_t it = 0;
#pragma unroll 1
    for (int tile = blockIdx.x; tile < P.n_tiles; tile += gridDim.x, ++it) {
        const int lane0 = tile * W + w0;
        float2* dst = P.out + (size_t)tile * P.ly * W;
        mbar_wait(&bars[2], it & 1);
        if constexpr (C::PAIR) {
            PV pv;
#pragma unroll
            for (int e = 0; e < 16; ++e) {
                if (e < NE) {
                    const ulonglong2 t2 = reinterpret_cast<const ulonglong2*>(pf)[((u[0] + e * Q) * W + w0) >> 1];
                    pv.r[e] = t2.x; pv.i[e] = t2.y;
                } else {
                    pv.r[e] = pv.i[e] = 0ull;
                }
            }
            __syncthreads();                                 // everybody has its registers: the buffer is free
            if (threadIdx.x == 0 && tile + (int)gridDim.x < P.n_tiles) { fence_proxy_async(); fetch(tile + gridDim.x); }
            typename PipeMidSelect<LOGN, MID>::type mid(P, u, lane0, nullptr, 0);
            transform_p<LOGN, true, true, false>(pv, u[0], w0, sm, P.tw, mid, sy);
            ulonglong2* d2 = reinterpret_cast<ulonglong2*>(dst);
#pragma unroll
            for (int e = 0; e < NE; ++e) d2[((size_t)(u[0] + e * Q) * W + w0) >> 1] = make_ulonglong2(pv.r[e], pv.i[e]);
        } else {
            float2 v[2][16];
#pragma unroll
            for (int s = 0; s < 2; ++s)
#pragma unroll
                for (int e = 0; e < 16; ++e)
                    v[s][e] = (u[s] + e * Q < N / 2) ? pf[u[s] + e * Q] : make_float2(0.f, 0.f);
            __syncthreads();
            if (threadIdx.x == 0 && tile + (int)gridDim.x < P.n_tiles) { fence_proxy_async(); fetch(tile + gridDim.x); }
            typename MidSelect<LOGN, MID>::type mid{P, u, lane0, sm};
            transform<LOGN, true, true>(v, u, w0, sm, P.tw, mid, SyncCta());
#pragma unroll
            for (int s = 0; s < 2; ++s)
#pragma unroll
                for (int e = 0; e < 16; ++e)
                    if (u[s] + e * Q < N / 2) dst[u[s] + e * Q] = v[s][e];      // conj(field): see pass_kernel.cuh
        }
    }
}

template <int LOGN, int MID>
static cudaError_t launch_colpref(int n_tiles, cudaStream_t s, const PassParams& p) {
    constexpr size_t smem = Tile<LOGN>::SMEM_BYTES + 64 + PREFETCH_BYTES;
    DeviceInfo* d = device_info();
    if (!d) return cudaErrorInvalidDevice;
    const int n_sm = d->n_sm;
    static FuncOnce once;
    if (!once.done(d->index)) {
        cudaError_t e = cudaFuncSetAttribute(colpref_kernel<LOGN, MID>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        once.set(d->index);
    }
    PassParams q = p;
    q.n_tiles = n_tiles;
    colpref_kernel<LOGN, MID><<<n_tiles < n_sm ? n_tiles : n_sm, Tile<LOGN>::T, smem, s>>>(q);
    return cudaGetLastError();
}

}  // namespace cwo
