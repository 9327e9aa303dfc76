// pipe_kernel.cuh -- the streaming passes of pass_kernel.cuh as ONE persistent CTA per SM that keeps
// three tiles in flight: two 256-thread groups transform alternate tiles while the next tiles are
// already on their way from HBM into the third shared-memory buffer (cp.async.bulk / cp.async signalled
// through mbarriers).  Global loads therefore never stall the butterflies, and HBM always has ~64-128 KB
// of requests outstanding per SM.  Results leave straight from registers (128-bit stores).
//
//   tile j of this CTA = blockIdx.x + j * gridDim.x, handled by group j % 2 in buffer j % 3.
//   When a group has finished with the shared-memory image of tile j it issues the load of tile j + 3
//   into the same buffer (the other group will consume it), then stores its results.
//
// Same arithmetic and the same tile/unit mapping as pass_kernel.cuh (S3-S10 of SURVEY.md section 8(a));
// row passes always use the unit-pair mapping at the workspace side.
#pragma once
#include <stdint.h>

#include "pass_kernel.cuh"

namespace cwo {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* b, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* b, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
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
// global -> shared bulk copy (TMA, no tensor map), completion counted in bytes on the mbarrier
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void cp_async16(void* dst, const void* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
// the mbarrier receives one (pre-counted) arrival once all cp.async of this thread so far have landed
__device__ __forceinline__ void cp_async_arrive(uint64_t* bar) {
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// order this thread's generic-proxy accesses to shared memory before later async-proxy (bulk copy) writes
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

template <int LOGN, int KIND> struct PipeCfg {
    using C = Tile<LOGN>;
    static constexpr int GROUPS = 2, NBUF = 3, GT = 256;
    static constexpr size_t BUF_RAW = (KIND == ROW_FWD && C::SMEM_BYTES_X > C::SMEM_BYTES) ? C::SMEM_BYTES_X : C::SMEM_BYTES;
    static constexpr size_t BUF = (BUF_RAW + 127) / 128 * 128;
    static constexpr size_t SMEM = NBUF * BUF + 64;
    static constexpr bool CPASYNC = (KIND == ROW_INV);       // gather of 16-byte pieces; else bulk copies
    // ROW_FWD staging: row r of the tile at element r * (points + ROWPAD) (bank stagger between lane pairs)
    static constexpr int ROWPAD = C::W > 2 ? 16 / C::W : 0;
};

// Pipelined passes exist for the tile shapes that matter for HBM-sized fields: 256 threads per tile,
// lane pairs, W <= 8 (transform lengths 1024..4096): pipe_supported() in pass_kernel.cuh.

template <int LOGN, int KIND, bool PAD, int MID, int IOM>
__global__ void __launch_bounds__(512, 1) pipe_kernel(const __grid_constant__ PassParams P) {
    using C = Tile<LOGN>;
    using K = PipeCfg<LOGN, KIND>;
    static_assert(C::T == K::GT && C::PAIR && C::W <= 8, "tile shape");
    constexpr int W = C::W, Q = C::Q, N = C::N;
    constexpr int NE = PAD ? 8 : 16;           // PAD: points >= n/2 are zero on load / dropped on store
    constexpr int NP = PAD ? N / 2 : N;        // points per lane that exist in memory at the padded side
    extern __shared__ __align__(128) unsigned char smraw[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smraw + K::NBUF * K::BUF);

    const int g = threadIdx.x >> 8, t = threadIdx.x & 255;
    const SyncGroup sync{1 + g};
    const int nt = (P.n_tiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;   // tiles of this CTA

    if (threadIdx.x == 0) {
#pragma unroll
        for (int b = 0; b < K::NBUF; ++b) mbar_init(&full[b], K::CPASYNC ? K::GT : 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // ---- load of tile j into buffer j % 3 (called by all 256 threads of one group) -------------------
    auto issue = [&](int j) {
        const int b = j % K::NBUF;
        const int tile = blockIdx.x + j * gridDim.x;
        unsigned char* dst = smraw + b * K::BUF;
        if constexpr (KIND == ROW_FWD) {
            // W rows of the row-major field, NP points each
            if (t == 0) {
                mbar_expect_tx(&full[b], W * NP * 8);
#pragma unroll
                for (int r = 0; r < W; ++r)
                    bulk_g2s(dst + (size_t)r * (NP + K::ROWPAD) * 8, P.in + (size_t)(tile * W + r) * P.pitch, NP * 8,
                             &full[b]);
            }
        } else if constexpr (KIND == ROW_INV) {
            // rows tile*W .. +W-1 of the column-tiled workspace: thread (w, i) fetches the 16-byte pieces
            // (points 2i + e*Q, +1 of row w) it will consume itself
            const int w = t % W, i2 = 2 * (t / W);
            const int row = tile * W + w;
            const int wcm = (1 << P.logwc) - 1;
#pragma unroll
            for (int e = 0; e < 16; ++e) {
                const int x = i2 + e * Q;
                const size_t a = (((size_t)(x >> P.logwc) * P.ly + row) << P.logwc) + (x & wcm);
                cp_async16(dst + (size_t)(e * K::GT + t) * 16, P.in + a);
            }
            cp_async_arrive(&full[b]);
        } else {
            // column tile: one contiguous [ly][W] block
            if (t == 0) {
                const uint32_t bytes = (uint32_t)P.ly * W * 8;
                mbar_expect_tx(&full[b], bytes);
                const unsigned char* src = reinterpret_cast<const unsigned char*>(P.in + (size_t)tile * P.ly * W);
                constexpr uint32_t CH = 16384;
                for (uint32_t o = 0; o < bytes; o += CH) bulk_g2s(dst + o, src + o, bytes - o < CH ? bytes - o : CH, &full[b]);
            }
        }
    };

    if (g == 0) {
        if (nt > 0) issue(0);
        if (nt > 2) issue(2);
    } else {
        if (nt > 1) issue(1);
    }

    const int us = t / (W / 2), w0 = 2 * (t % (W / 2));     // standard mapping: unit us, lanes w0, w0+1
    const int u[2] = {us, us};
    const int xw = t % W, xi2 = 2 * (t / W);                // unit-pair mapping: lane xw, units xi2, xi2+1

#pragma unroll 1
    for (int j = g; j < nt; j += K::GROUPS) {
        const int b = j % K::NBUF;
        const int tile = blockIdx.x + j * gridDim.x;
        float2* sm = reinterpret_cast<float2*>(smraw + b * K::BUF);
        float2 v[2][16];
        mbar_wait(&full[b], (j / K::NBUF) & 1);

        // ---- registers <- staged tile ------------------------------------------------------------
        if constexpr (KIND == ROW_FWD) {
#pragma unroll
            for (int s = 0; s < 2; ++s)
#pragma unroll
                for (int e = 0; e < 16; ++e)
                    v[s][e] = (e < NE) ? sm[(w0 + s) * (NP + K::ROWPAD) + us + e * Q] : make_float2(0.f, 0.f);
        } else if constexpr (KIND == ROW_INV) {
#pragma unroll
            for (int e = 0; e < 16; ++e) {
                const float4 t4 = reinterpret_cast<const float4*>(sm)[e * K::GT + t];
                v[0][e] = make_float2(t4.x, -t4.y); v[1][e] = make_float2(t4.z, -t4.w);
            }
        } else {
#pragma unroll
            for (int e = 0; e < 16; ++e) {
                if (e < NE) {
                    const float4 t4 = *reinterpret_cast<const float4*>(&sm[(us + e * Q) * W + w0]);
                    v[0][e] = make_float2(t4.x, t4.y); v[1][e] = make_float2(t4.z, t4.w);
                } else {
                    v[0][e] = v[1][e] = make_float2(0.f, 0.f);
                }
            }
        }

        // ---- transform (the first barrier inside also retires the staged image) ------------------
        const int lane0 = tile * W + w0;
        if constexpr (KIND == ROW_FWD) {
            transform_fwd_xlast<LOGN>(v, t, sm, P.tw, sync);
        } else if constexpr (KIND == ROW_INV) {
            transform_inv_xfirst<LOGN>(v, t, sm, P.tw, sync);
        } else if constexpr (KIND == COL_FWD) {
            transform<LOGN, true, false>(v, u, w0, sm, P.tw, MidNone(), sync);
        } else {
            typename MidSelect<LOGN, MID>::type mid{P, u, lane0, sm};
            if constexpr (KIND == COL_FUSED) {
                transform<LOGN, true, true>(v, u, w0, sm, P.tw, mid, sync);
            } else {
                mid(v);
                transform<LOGN, false, true>(v, u, w0, sm, P.tw, MidNone(), sync);
            }
        }

        // ---- this buffer is free: fetch tile j + 3 into it ----------------------------------------
        fence_proxy_async();
        sync();
        if (j + K::NBUF < nt) issue(j + K::NBUF);

        // ---- store (conj completes an inverse transform) ------------------------------------------
        if constexpr (KIND == ROW_FWD) {
            const int row = tile * W + xw;
            const int wcm = (1 << P.logwc) - 1;
#pragma unroll
            for (int e = 0; e < 16; ++e) {
                const int x = xi2 + e * Q;
                const size_t a = (((size_t)(x >> P.logwc) * P.ly + row) << P.logwc) + (x & wcm);
                *reinterpret_cast<float4*>(&P.out[a]) = make_float4(v[0][e].x, v[0][e].y, v[1][e].x, v[1][e].y);
            }
        } else if constexpr (KIND == ROW_INV) {
            static_assert(IOM == OUT_COMPLEX, "GS store modes run in pass_kernel");
            const float sc = P.out_scale;
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                float2* dst = P.out + (size_t)(tile * W + w0 + s) * P.pitch + us;
#pragma unroll
                for (int e = 0; e < NE; ++e) dst[e * Q] = make_float2(v[s][e].x * sc, -v[s][e].y * sc);
            }
        } else {
            float2* dst = P.out + (size_t)tile * P.ly * W;
            constexpr bool CONJ = (KIND != COL_FWD);
#pragma unroll
            for (int e = 0; e < NE; ++e) {
                const float2 a = v[0][e], c = v[1][e];
                *reinterpret_cast<float4*>(&dst[(size_t)(us + e * Q) * W + w0]) =
                    CONJ ? make_float4(a.x, -a.y, c.x, -c.y) : make_float4(a.x, a.y, c.x, c.y);
            }
        }
    }
}

template <int LOGN, int KIND, bool PAD, int MID, int IOM>
static cudaError_t launch_pipe(int n_tiles, cudaStream_t s, const PassParams& p) {
    using K = PipeCfg<LOGN, KIND>;
    static int n_sm = 0;
    if (!n_sm) {
        int dev = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) return e;
        e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return e;
    }
    static bool configured = false;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(pipe_kernel<LOGN, KIND, PAD, MID, IOM>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, (int)K::SMEM);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    PassParams q = p;
    q.n_tiles = n_tiles;
    const int grid = n_tiles < n_sm ? n_tiles : n_sm;
    pipe_kernel<LOGN, KIND, PAD, MID, IOM><<<grid, 512, K::SMEM, s>>>(q);
    return cudaGetLastError();
}

}  // namespace cwo
