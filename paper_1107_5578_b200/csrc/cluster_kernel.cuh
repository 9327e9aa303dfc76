// cluster_kernel.cuh -- forward row pass (R) for 16384-point rows on a 4-CTA thread-block cluster.
//
// A 16384-point row is one 139 KB tile, one CTA per SM, and with single-lane column tiles (Wc = 1) the workspace
// is plain column-major T[x][y]: a row tile owns ONE row, so its results go out as 16384 pieces of 8 bytes, a
// quarter of a DRAM sector each.  Measured on the 8192^2 Fresnel propagation: that scatter is 965 us of the pass's
// 1514 us (scattered partial-sector writes cost the memory system a request each, see fold_kernel.cuh).
// Here the four CTAs of a cluster transform four consecutive rows y0..y0+3, stage their results in their own
// shared memory as [owner][column], and then every CTA o READS, through distributed shared memory and fully
// coalesced, the block [o] of all four CTAs: columns [4096 o, 4096 (o+1)) of all four rows.  It rewrites them as
// [column][4 rows], one full 32-byte sector per column, and stores its quarter with TMA tensor copies (box
// 32 B x 256 columns).  (Pushing the results with scattered 8-byte st.shared::cluster instead was measured
// slower than the plain kernel: 1727 us.)  Loads and the transform are those of pass_kernel.cuh (ROW_FWD).
// Pass 1514 -> 1024 us.  The mirrored inverse pass (TMA gather of 32-byte pieces, rows redistributed through
// distributed shared memory) was built and measured as well and is not used: 8-byte GATHERS are not what bounds
// pass R' (1056 -> 1130 us).
#pragma once
#include "pipe_kernel.cuh"

namespace cwo {

__device__ __forceinline__ uint32_t cluster_ctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// 8-byte load from the shared memory of CTA `rank` of the cluster, at the address that `local` has in ours
__device__ __forceinline__ float2 ld_cluster_f2(const void* local, uint32_t rank) {
    uint32_t ra;
    float2 v;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(ra) : "r"(smem_u32(local)), "r"(rank));
    asm volatile("ld.shared::cluster.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(ra) : "memory");
    return v;
}

constexpr int CLUSTER_ROWS = 4;

// P.tmap: the workspace T[x][y] as a 2-D float tensor {2 Ny, Mx} with boxes of 4 rows (8 floats) x 256 columns.
template <int LOGN, bool PAD>
__global__ void __launch_bounds__(Tile<LOGN>::T, 1) cluster_row_fwd_kernel(const __grid_constant__ PassParams P) {
    using C = Tile<LOGN>;
    static_assert(!C::PAIR && C::W == 1, "one lane per tile");
    constexpr int Q = C::Q, N = C::N, T = C::T, NE = PAD ? 8 : 16, COLS = N / CLUSTER_ROWS, CPT = COLS / T;
    static_assert(sizeof(float2) * N <= C::SMEM_BYTES && COLS % T == 0, "staging fits the tile buffer");
    extern __shared__ float2 sm[];
    const uint32_t rank = cluster_ctarank();                // clusters are 4 consecutive CTAs
    const int u[2] = {(int)threadIdx.x, (int)threadIdx.x + Q / 2};
    // Persistent over row quads (the grid is one wave of clusters): the TMA store of one quad reads the tile buffer
    // while the next quad's rows are loaded from global memory.
#pragma unroll 1
    for (int row = blockIdx.x; row < P.n_tiles; row += gridDim.x) {
    float2 v[2][16];
#pragma unroll
    for (int s = 0; s < 2; ++s) {
        const size_t base = (size_t)row * P.pitch + u[s];
#pragma unroll
        for (int e = 0; e < 16; ++e) v[s][e] = (e < NE) ? P.in[base + e * Q] : make_float2(0.f, 0.f);
    }
    if (row != (int)blockIdx.x) {                           // the previous quad's store has read the tile buffer
        if (threadIdx.x == 0) bulk_wait_read();
        __syncthreads();
    }
    transform<LOGN, true, false>(v, u, 0, sm, P.tw, MidNone(), SyncCta());
    // register e of slot s <-> point (column) p = u[s] + e*Q of this row; stage as [owner p / COLS][p % COLS] = sm[p]
    __syncthreads();                                        // tile buffer no longer being read
#pragma unroll
    for (int s = 0; s < 2; ++s)
#pragma unroll
        for (int e = 0; e < 16; ++e) sm[u[s] + e * Q] = v[s][e];
    cluster_sync();                                         // the four rows are staged
    float2 g[CPT][CLUSTER_ROWS];                            // my columns c = t + T k of the four rows
#pragma unroll
    for (int k = 0; k < CPT; ++k)
#pragma unroll
        for (int rr = 0; rr < CLUSTER_ROWS; ++rr)
            g[k][rr] = ld_cluster_f2(&sm[rank * COLS + threadIdx.x + T * k], (uint32_t)rr);
    cluster_sync();                                         // everybody has read everybody's staging
#pragma unroll
    for (int k = 0; k < CPT; ++k) {
        float4* d = reinterpret_cast<float4*>(&sm[(threadIdx.x + T * k) * CLUSTER_ROWS]);
        d[0] = make_float4(g[k][0].x, g[k][0].y, g[k][1].x, g[k][1].y);
        d[1] = make_float4(g[k][2].x, g[k][2].y, g[k][3].x, g[k][3].y);
    }
    fence_proxy_async();
    __syncthreads();
    if (threadIdx.x == 0) {
        const int row0 = row - (int)rank;
        for (int b = 0; b < COLS / 256; ++b)
            tma_store_2d(&P.tmap, sm + (size_t)b * 256 * CLUSTER_ROWS, row0 * 2, (int)rank * COLS + b * 256);
        bulk_commit();
    }
    }   // row quads
    if (threadIdx.x == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}

template <int LOGN, bool PAD>
static cudaError_t launch_cluster_row_fwd(int n_rows, cudaStream_t s, const PassParams& p) {
    constexpr size_t smem = Tile<LOGN>::SMEM_BYTES + 64;
    DeviceInfo* d = device_info();
    if (!d) return cudaErrorInvalidDevice;
    static FuncOnce once;
    if (!once.done(d->index)) {
        cudaError_t e = cudaFuncSetAttribute(cluster_row_fwd_kernel<LOGN, PAD>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)smem);
        if (e != cudaSuccess) return e;
        once.set(d->index);
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)n_rows); cfg.blockDim = dim3((unsigned)Tile<LOGN>::T);
    cfg.dynamicSmemBytes = smem; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = CLUSTER_ROWS; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    static std::atomic<int> waves[MAX_DEVICES];             // CTAs of the clusters that are resident at once, per device
    int wave = waves[d->index].load(std::memory_order_acquire);
    if (!wave) {
        int nc = 0;
        cudaError_t e = cudaOccupancyMaxActiveClusters(&nc, cluster_row_fwd_kernel<LOGN, PAD>, &cfg);
        if (e != cudaSuccess) return e;
        wave = (nc > 0 ? nc : 1) * CLUSTER_ROWS;
        waves[d->index].store(wave, std::memory_order_release);
    }
    if (n_rows > wave) cfg.gridDim = dim3((unsigned)wave);
    PassParams q = p;
    q.n_tiles = n_rows;
    return cudaLaunchKernelEx(&cfg, cluster_row_fwd_kernel<LOGN, PAD>, q);
}

}  // namespace cwo
