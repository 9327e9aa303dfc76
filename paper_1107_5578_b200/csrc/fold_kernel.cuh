// fold_kernel.cuh -- pipelined INVERSE row pass (R') for transform length 2n = 8192 (and zero-expanded 4096), built on
// the n-point tile of pipe_kernel.cuh: one row is FOLDED into the two slots of a thread.
//
// A tile of two 8192-point lanes no longer fits three times in shared memory, so the 8192-point passes of
// pass_kernel.cuh run one 139 KB tile per SM with nothing overlapped.  One radix-2 step (decimation in time,
// forward kernel on the conjugated data as everywhere, see pass_kernel.cuh) removes the problem:
//       A = FFT_n(X[even]),  B = FFT_n(X[odd]);  y[x] = A[x] + w^x B[x],  y[x+n] = A[x] - w^x B[x],  w = exp(-i 2 pi/2n)
// X[even], X[odd] are two ordinary n-point lanes with the SAME twiddles: exactly the lane pair (slot 0, slot 1)
// of the 4096-point tile, and X[2k], X[2k+1] are neighbouring columns of the row, i.e. one planar 16-byte
// element of the column-tiled workspace -- no unit-pair mapping is needed.  The tile is ONE row (64 KB, three
// buffers); the radix-2 step runs in registers while the row is written to its row-major staging.
// Zero padding (Fresnel): y[x+n] is not formed.
// Measured (8192^2 ASM): 443 -> 280 us.  The mirrored forward pass (decimation in frequency) was built and
// measured too and is NOT used: its workspace side writes 16-byte pieces, half a DRAM sector each, and scattered
// partial-sector writes run at about half the rate of the 32-byte pieces the two-row tiles of pass R write
// (641 us with TMA stores, 745 us with st.global, against 350 us).
// Same producer / consumer-group / mbarrier structure as pipe_kernel.cuh; transform = the packed lane pair of
// fft_packed.cuh (round 2; the scalar ping-pong form of pp_core.cuh took 277 us at 8192^2).
#pragma once
#include "pipe_kernel.cuh"

namespace cwo {

template <int LOGC> struct FoldCfg {
    using C = Tile<LOGC>;
    // one row = the lane pair (even columns, odd columns) of the n-point transform: n/16 threads; 512 consumer threads
    // per CTA in groups of one row each, and as many row buffers as fit (n = 4096: 2 groups, 3 buffers of 70 KB;
    // n = 2048: 4 groups, 6 buffers of 35 KB)
    static constexpr int GT = C::Q, GROUPS = 512 / GT, NBUF = GROUPS + GROUPS / 2;
    static constexpr int THREADS = GROUPS * GT + 128;
    static constexpr size_t BUF = (sizeof(float2) * (size_t)(C::N + C::N / 16) * 2 + 127) / 128 * 128;   // >= one row (16 n bytes)
    static constexpr int NTW = PP<LOGC>::NTW_P;
    static constexpr size_t TW_OFF = NBUF * BUF + 128;                         // n-point stage twiddles
    static constexpr size_t TW2_OFF = TW_OFF + sizeof(float2) * NTW;           // 2n-point twiddles w^us, us < Q
    static constexpr size_t SMEM = TW2_OFF + sizeof(float2) * C::Q;
    static_assert(GT == 128 || GT == 256, "rows of 4096 or 8192 points");
    static_assert(BUF >= sizeof(float2) * 2 * C::N, "row staging fits the tile buffer");
    static_assert(2 * NBUF * sizeof(uint64_t) <= 128, "mbarriers fit their slot");
};

// barrier over the GT threads of one row group
template <int GT> struct SyncRow {
    static constexpr bool EARLY_WAR = false;
    int id;
    __device__ __forceinline__ void operator()() const { asm volatile("bar.sync %0, %1;" ::"r"(id), "n"(GT) : "memory"); }
    __device__ __forceinline__ void consumed() const {}
    __device__ __forceinline__ void war() const { (*this)(); }
    __device__ __forceinline__ void raw() const { (*this)(); }
    __device__ __forceinline__ void raw_arrive() const {}
    __device__ __forceinline__ void raw_wait() const { (*this)(); }
};

// Pass R': workspace -> IFFT_2n -> u2.
// P.tw: the 2n-point twiddle table.  P.tmap: the workspace with boxes of ONE row (16 bytes x 256 column pairs).
template <int LOGC, bool PAD>
__global__ void __launch_bounds__(FoldCfg<LOGC>::THREADS, 1) fold_row_kernel(const __grid_constant__ PassParams P) {
    using C = Tile<LOGC>;
    using K = FoldCfg<LOGC>;
    constexpr int Q = C::Q, N = C::N;
    constexpr int NPR = PAD ? N : 2 * N;                    // points of a row that exist in the row-major field
    constexpr int GR = N / 256;                             // TMA boxes (256 column pairs each) per row
    constexpr int GT = K::GT;
    extern __shared__ __align__(128) unsigned char smraw[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smraw + K::NBUF * K::BUF);
    uint64_t* staged = full + K::NBUF;
    const int nt = (P.n_tiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;

    if (threadIdx.x == 0) {
#pragma unroll
        for (int b = 0; b < K::NBUF; ++b) { mbar_init(&full[b], 1); mbar_init(&staged[b], K::GT); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    float2* tws = reinterpret_cast<float2*>(smraw + K::TW_OFF);
    float2* tw2 = reinterpret_cast<float2*>(smraw + K::TW2_OFF);
    for (int i = threadIdx.x; i < K::NTW; i += K::THREADS) tws[i] = __ldg(&P.tw[2 * i]);
    for (int i = threadIdx.x; i < Q; i += K::THREADS) tw2[i] = __ldg(&P.tw[i]);
    asm volatile("griddepcontrol.wait;" ::: "memory");      // see pipe_kernel.cuh
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    __syncthreads();

    if (threadIdx.x >= K::GROUPS * K::GT) {
        // ================================ producer warp (one lane) ================================
        asm volatile("setmaxnreg.dec.sync.aligned.u32 24;");
        if (threadIdx.x != K::GROUPS * K::GT) return;
        auto load = [&](int j) {                            // the row's 16-byte elements, one per column pair
            const int b = j % K::NBUF, row = blockIdx.x + j * gridDim.x;
            unsigned char* dst = smraw + b * K::BUF;
            mbar_expect_tx(&full[b], 2 * N * 8);
            for (int c = 0; c < GR; ++c) tma_load_2d(dst + (size_t)c * 256 * 16, &P.tmap, row * 4, c * 256, &full[b]);
        };
        auto store = [&](int j) {                           // one row of the row-major field
            const int b = j % K::NBUF, row = blockIdx.x + j * gridDim.x;
            const unsigned char* src = smraw + b * K::BUF;
            unsigned char* dst = reinterpret_cast<unsigned char*>(P.out + (size_t)row * P.pitch);
            for (uint32_t o = 0; o < NPR * 8u; o += 16384u) bulk_s2g(dst + o, src + o, 16384u);
            bulk_commit();
        };
        for (int j = 0; j < nt && j < K::NBUF; ++j) load(j);
        for (int j = 0; j < nt; ++j) {
            mbar_wait_backoff(&staged[j % K::NBUF], (j / K::NBUF) & 1);
            store(j);
            if (j + K::NBUF < nt) { bulk_wait_read(); load(j + K::NBUF); }
        }
        asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
        return;
    }

    // ===================================== consumer groups =====================================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 112;");
    const int g = threadIdx.x / GT, us = threadIdx.x % GT;
    const SyncRow<GT> sync{1 + g};
    const float2 wb = tw2[us];                              // w^us
#pragma unroll 1
    for (int j = g; j < nt; j += K::GROUPS) {
        const int b = j % K::NBUF;
        float2* sm = reinterpret_cast<float2*>(smraw + b * K::BUF);
        PV pv;
        mbar_wait(&full[b], (j / K::NBUF) & 1);
        // one planar element per column pair: (re X[2k], re X[2k+1], im X[2k], im X[2k+1]), k = us + e*Q = the packed
        // register pair (slot 0 = even columns, slot 1 = odd columns); the column pass left conj(field) here
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            const ulonglong2 t2 = *reinterpret_cast<const ulonglong2*>(&sm[2 * (us + e * Q)]);
            pv.r[e] = t2.x; pv.i[e] = t2.y;
        }
        sync();                                             // staged image retired
        transform_p<LOGC, false, true, false, MidNone, SyncRow<GT>, 1>(pv, us, 0, sm, tws, MidNone(), sync);
        sync();                                             // nobody still reads the exchange image
        const float sc = P.out_scale;                       // conj completes the inverse transform
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            float ar, br, ai, bi;
            pk_split(pv.r[e], ar, br); pk_split(pv.i[e], ai, bi);
            const float2 t = cmul(make_float2(br, bi), cmul(wb, w32_pow(e)));   // w^x B[x], x = us + e*Q
            sm[us + e * Q] = make_float2((ar + t.x) * sc, -(ai + t.y) * sc);
            if constexpr (!PAD) sm[N + us + e * Q] = make_float2((ar - t.x) * sc, -(ai - t.y) * sc);
        }
        fence_proxy_async();
        mbar_arrive(&staged[b]);
    }
}

template <int LOGC, bool PAD>
static cudaError_t launch_fold(int n_rows, cudaStream_t s, const PassParams& p) {
    using K = FoldCfg<LOGC>;
    DeviceInfo* d = device_info();
    if (!d) return cudaErrorInvalidDevice;
    const int n_sm = d->n_sm;
    static FuncOnce once;
    if (!once.done(d->index)) {
        cudaError_t e = cudaFuncSetAttribute(fold_row_kernel<LOGC, PAD>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)K::SMEM);
        if (e != cudaSuccess) return e;
        once.set(d->index);
    }
    PassParams q = p;
    q.n_tiles = n_rows;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(n_rows < n_sm ? n_rows : n_sm)); cfg.blockDim = dim3((unsigned)K::THREADS);
    cfg.dynamicSmemBytes = K::SMEM; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, fold_row_kernel<LOGC, PAD>, q);
}

}  // namespace cwo
