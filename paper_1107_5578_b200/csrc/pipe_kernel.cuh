// pipe_kernel.cuh -- the streaming passes of pass_kernel.cuh as ONE persistent, warp-specialised CTA per
// SM that keeps three tiles in flight in three shared-memory buffers:
//   * two 256-thread consumer groups transform alternate tiles (tile j of this CTA = blockIdx.x +
//     j * gridDim.x, group j % 2, buffer j % 3); they touch global memory only for twiddles/tables;
//   * one producer warp moves every tile: TMA bulk / tensor loads into a buffer (mbarrier full[b]),
//     and, once the group has written its results back into the same buffer in the layout of the
//     destination (mbarrier staged[b]), TMA bulk / tensor stores out of it, then the load of tile j + 3.
// HBM therefore always has 64-192 KB of requests outstanding per SM, none of them waiting on a
// butterfly, and the 32-byte scatter/gather of the column-tiled workspace never occupies the SM's
// load/store path.
//
// Same arithmetic and the same tile/unit mapping as pass_kernel.cuh (S3-S10 of SURVEY.md section 8(a));
// row passes always use the unit-pair mapping at the workspace side and run the scalar ping-pong schedule
// of pp_core.cuh; column passes run both slots of a thread in lockstep on packed f32x2 operands
// (fft_packed.cuh), fed directly by the planar lane-pair layout of the workspace.
// The twiddles every stage needs, and the ASM theta_y table, are copied to shared memory once per CTA.
#pragma once
#include <stdint.h>

#include "pass_kernel.cuh"

#ifndef CWO_SETMAXNREG
#define CWO_SETMAXNREG 1
#endif

namespace cwo {


// same, for the producer lane: back off between polls so that the spin does not take issue slots from the
// four consumer warps that share its scheduler
__device__ __forceinline__ void mbar_wait_backoff(uint64_t* b, uint32_t parity) {
    uint32_t ok;
    for (;;) {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(ok)
            : "r"(smem_u32(b)), "r"(parity)
            : "memory");
        if (ok) break;
        __nanosleep(64);
    }
}
__device__ __forceinline__ void cp_async16(void* dst, const void* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
// the mbarrier receives one (pre-counted) arrival once all cp.async of this thread so far have landed
__device__ __forceinline__ void cp_async_arrive(uint64_t* bar) {
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// shared -> global tensor store of one box (2-D), bulk-group completion
__device__ __forceinline__ void tma_store_2d(const CUtensorMap* m, const void* src, int c0, int c1) {
    asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%2, %3}], [%1];" ::"l"(m),
                 "r"(smem_u32(src)), "r"(c0), "r"(c1)
                 : "memory");
}
// global -> shared tensor load of one box (2-D), completion counted in bytes on the mbarrier
__device__ __forceinline__ void tma_load_2d(void* dst, const CUtensorMap* m, int c0, int c1, uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];" ::"r"(
            smem_u32(dst)),
        "l"(m), "r"(smem_u32(bar)), "r"(c0), "r"(c1)
        : "memory");
}
// shared -> global bulk copy (contiguous), bulk-group completion
__device__ __forceinline__ void bulk_s2g(void* dst, const void* src, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(smem_u32(src)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
// all bulk stores of this thread have finished READING shared memory
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }

// Mid functors with a packed() form (both slots of a thread, fft_packed.cuh); tables that do not depend on the tile come
// from shared memory, the per-lane values are fetched when the functor is built (top of the tile).
template <int LOGN> struct PipeMidAsmSplit {
    using C = Tile<LOGN>;
    const PassParams& P; const float* thy; int us, lane0; float thx[2], res_c;
    // plane > 0 or batched: the plane's tables are read from global memory (thy_ == nullptr)
    __device__ __forceinline__ PipeMidAsmSplit(const PassParams& P_, const int (&u)[2], int lane0_, const float* thy_,
                                               int plane = 0)
        : P(P_), thy(thy_), us(u[0]), lane0(lane0_), res_c(P_.res_c) {
        const float* thl = reinterpret_cast<const float*>(P.tab_lane) + (size_t)plane * P.tab_plane_stride;
        if (!thy_) {
            thy = reinterpret_cast<const float*>(P.tab_point) + (size_t)plane * P.tab_plane_stride;
            if (P.plane_resc) res_c = __ldg(&P.plane_resc[plane]);
        }
        const float2 t = __ldg(reinterpret_cast<const float2*>(&thl[lane0]));     // lane0 is even
        thx[0] = t.x; thx[1] = t.y;
    }
    // Both slots in packed form (fft_packed.cuh).  z sqrt(1/lambda^2 - f^2) = (z/lambda)(1 - s/2 - g(s)),
    // g(s) = s^2/8 + s^3/16 + 5 s^4/128 + 7 s^5/256 + 21 s^6/1024 + 33 s^7/2048 + ...: when the plan has verified that
    // the truncated series is exact to 1e-7 cycles for every bin (P.res_poly) the residual is that polynomial in
    // packed arithmetic (the two slots differ in s only; theta_y, s_y broadcast), reduced mod 1 BEFORE it meets the
    // table phases (so the sum keeps 6e-8-cycle resolution), and the only scalar work left is the sine and cosine;
    // otherwise the closed form with rsqrt / division per sample.
    // Eq.(18): the two Rect band limits (CWO_OPT_ASM_BAND_LIMIT); uniform branch, off by default
    __device__ __forceinline__ void band_mask(PV& v) const {
        const int n = P.n_lane_bins;
        const int k0 = (lane0 < n / 2) ? lane0 : lane0 - n, k1 = (lane0 + 1 < n / 2) ? lane0 + 1 : lane0 + 1 - n;
        const bool c0 = k0 < P.band_lane_lo || k0 > P.band_lane_hi, c1 = k1 < P.band_lane_lo || k1 > P.band_lane_hi;
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            const int l = us + e * C::Q;
            const int ls = (l < C::N / 2) ? l : l - C::N;
            const bool cp = ls < P.band_point_lo || ls > P.band_point_hi;
            float r0, r1, i0, i1;
            pk_split(v.r[e], r0, r1); pk_split(v.i[e], i0, i1);
            if (cp || c0) { r0 = 0.f; i0 = 0.f; }
            if (cp || c1) { r1 = 0.f; i1 = 0.f; }
            v.r[e] = pk_make(r0, r1); v.i[e] = pk_make(i0, i1);
        }
    }
    __device__ __forceinline__ void packed(PV& v) const {
        if (P.res_poly) packed_poly(v); else packed_closed(v);
        if (P.band) band_mask(v);
    }
    __device__ __forceinline__ void packed_poly(PV& v) const {
        float sx[2];
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            const int lane = lane0 + s;
            const int ks = (lane < P.n_lane_bins / 2) ? lane : lane - P.n_lane_bins;
            sx[s] = P.res_a * (float)ks * (float)ks;
        }
        const pk sx2 = pk_make(sx[0], sx[1]), thx2 = pk_make(thx[0], thx[1]);
        const float usf = (float)us;
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            const int l = us + e * C::Q;
            const float lsf = usf + (float)(e < 8 ? e * C::Q : (e - 16) * C::Q);   // signed bin of l (us < Q), exact
            const float sy = P.res_b * lsf * lsf;
            const pk sv = add2(sx2, pk_bcast(sy));
            pk h = fma2(sv, pk_bcast(33.0f / 2048.0f), pk_bcast(21.0f / 1024.0f));
            h = fma2(sv, h, pk_bcast(7.0f / 256.0f));
            h = fma2(sv, h, pk_bcast(5.0f / 128.0f));
            h = fma2(sv, h, pk_bcast(1.0f / 16.0f));
            h = fma2(sv, h, pk_bcast(0.125f));
            pk res = mul2(mul2(mul2(sv, sv), pk_bcast(res_c)), h);
            const pk big = pk_bcast(12582912.0f);                  // 1.5 * 2^23: (x + big) - big = rint(x), |x| < 2^22
            res = sub2(res, sub2(add2(res, big), big));
            const pk ph = mul2(sub2(add2(thx2, pk_bcast(thy[l])), res), pk_bcast(6.283185307179586f));
            float p0, p1, sn0, cs0, sn1, cs1;
            pk_split(ph, p0, p1);
            __sincosf(p0, &sn0, &cs0); __sincosf(p1, &sn1, &cs1);
            // conj(x (cs + i sn)) = (xr cs - xi sn) - i (xr sn + xi cs)
            const pk cs2 = pk_make(cs0, cs1), sn2 = pk_make(sn0, sn1), xr = v.r[e], xi = v.i[e];
            v.r[e] = fma2(xr, cs2, pk_neg(mul2(xi, sn2)));
            v.i[e] = fma2(pk_neg(xr), sn2, pk_neg(mul2(xi, cs2)));
        }
    }
    __device__ __forceinline__ void packed_closed(PV& v) const {
        float sx[2];
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            const int lane = lane0 + s;
            const int ks = (lane < P.n_lane_bins / 2) ? lane : lane - P.n_lane_bins;
            sx[s] = P.res_a * (float)ks * (float)ks;
        }
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            const int l = us + e * C::Q;
            const int ls = (l < C::N / 2) ? l : l - C::N;
            const float ty = thy[l], sy = P.res_b * (float)ls * (float)ls;
            float xr[2], xi[2];
            pk_split(v.r[e], xr[0], xr[1]); pk_split(v.i[e], xi[0], xi[1]);
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                const float sv = sy + sx[s];
                const float om = 1.0f - sv;
                const float r = 1.0f + om * rsqrtf(om);
                const float res = __fdividef(res_c * sv * sv, 2.0f * r * r);
                float ph = thx[s] + ty - res;
                ph -= rintf(ph);
                float sn, cs;
                __sincosf(6.283185307179586f * ph, &sn, &cs);
                const float2 y = cmul(make_float2(xr[s], xi[s]), make_float2(cs, sn));
                xr[s] = y.x; xi[s] = -y.y;
            }
            v.r[e] = pk_make(xr[0], xr[1]); v.i[e] = pk_make(xi[0], xi[1]);
        }
    }
};
template <int LOGN> struct PipeMidTables : MidTables<LOGN> {
    __device__ __forceinline__ PipeMidTables(const PassParams& P, const int (&u)[2], int lane0, const float*, int = 0)
        : MidTables<LOGN>{P, u, lane0, nullptr} {}
};
struct PipeMidNone : MidNone {
    __device__ __forceinline__ PipeMidNone(const PassParams&, const int (&)[2], int, const float*, int = 0) {}
};
template <int LOGN, int MID> struct PipeMidSelect;
template <int LOGN> struct PipeMidSelect<LOGN, MID_NONE> { using type = PipeMidNone; };
template <int LOGN> struct PipeMidSelect<LOGN, MID_TABLES> { using type = PipeMidTables<LOGN>; };
template <int LOGN> struct PipeMidSelect<LOGN, MID_ASM_SPLIT> { using type = PipeMidAsmSplit<LOGN>; };

template <int LOGN, int KIND> struct PipeCfg {
    using C = Tile<LOGN>;
#ifndef CWO_GROUPS
#define CWO_GROUPS 2
#endif
    static constexpr int GROUPS = CWO_GROUPS, NBUF = 3, GT = 256;
    // + the producer: a warpgroup that hands its registers over (setmaxnreg: 112 / 24 per thread), or just one warp
    // with the register file split evenly (65536 / 544 = 120 per thread)
    static constexpr int THREADS = GROUPS * GT + (CWO_SETMAXNREG ? 128 : 32);
    static constexpr size_t BUF_RAW = (KIND == ROW_FWD && C::SMEM_BYTES_X > C::SMEM_BYTES) ? C::SMEM_BYTES_X : C::SMEM_BYTES;
    static constexpr size_t BUF = (BUF_RAW + 127) / 128 * 128;
    static constexpr size_t TW_OFF = NBUF * BUF + 64;                       // after the mbarriers
    // full-length stage twiddles, then (packed row passes) the half-length ones, tw_h[i] = tw_n[2i]
    static constexpr int NTW_H = PP<LOGN - 1>::NTW_P;
    static constexpr size_t TW_BYTES = sizeof(float2) * (PP<LOGN>::NTW + NTW_H);
    static constexpr size_t TAB_OFF = TW_OFF + TW_BYTES;                    // ASM: theta_y[l] (float, N entries)
    static constexpr size_t TAB_BYTES = sizeof(float) * C::N;
    static constexpr size_t SMEM_NOTAB = TAB_OFF, SMEM_TAB = TAB_OFF + TAB_BYTES;
    // row-major staging (ROW_FWD in, ROW_INV out): row r of the tile at element r * (points + ROWPAD)
    // (bank stagger between lane pairs)
    static constexpr int ROWPAD = 16 / C::W;              // (W = 2: the packed row passes read rows r, r+1 from neighbouring threads)
};

// Pipelined passes exist for the tile shapes that matter for HBM-sized fields: 256 threads per tile,
// lane pairs, W <= 8 (transform lengths 1024..4096): pipe_supported() in pass_kernel.cuh.

template <int LOGN, int KIND, bool PAD, int MID, int IOM>
#if CWO_SETMAXNREG
__global__ void __launch_bounds__(PipeCfg<LOGN, KIND>::THREADS, 1)
#else
__global__ void __maxnreg__(120)
#endif
pipe_kernel(const __grid_constant__ PassParams P) {
    using C = Tile<LOGN>;
    using K = PipeCfg<LOGN, KIND>;
    static_assert(C::T == K::GT && C::PAIR && C::W <= 8, "tile shape");
    constexpr int W = C::W, Q = C::Q, N = C::N;
    constexpr int NE = PAD ? 8 : 16;           // PAD: points >= n/2 are zero on load / dropped on store
    constexpr int NP = PAD ? N / 2 : N;        // points per lane that exist in memory at the padded side
    constexpr int RS = NP + K::ROWPAD;         // row stride of the row-major staging
    extern __shared__ __align__(128) unsigned char smraw[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smraw + K::NBUF * K::BUF);   // tile landed in buffer b
    uint64_t* staged = full + K::NBUF;                                        // results written back to buffer b

    const int nt = (P.n_tiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;   // tiles of this CTA

    if (threadIdx.x == 0) {
#pragma unroll
        for (int b = 0; b < K::NBUF; ++b) { mbar_init(&full[b], 1); mbar_init(&staged[b], K::GT); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    // per-CTA copies of the small tables every tile needs (the L1 left beside ~220 KB of tile buffers is a few
    // KB: a global twiddle load would be an L2 round trip in the middle of every stage)
    float2* tws = reinterpret_cast<float2*>(smraw + K::TW_OFF);
    float* thy = reinterpret_cast<float*>(smraw + K::TAB_OFF);
    for (int i = threadIdx.x; i < PP<LOGN>::NTW; i += K::THREADS) tws[i] = __ldg(&P.tw[i]);
    float2* twh = tws + PP<LOGN>::NTW;
    if constexpr (KIND == ROW_FWD || KIND == ROW_INV)
        for (int i = threadIdx.x; i < K::NTW_H; i += K::THREADS) twh[i] = __ldg(&P.tw[2 * i]);
    const bool batched = P.n_planes > 1;
    if constexpr (MID == MID_ASM_SPLIT) {
        const float* thp = reinterpret_cast<const float*>(P.tab_point);
        if (!batched) for (int i = threadIdx.x; i < N; i += K::THREADS) thy[i] = __ldg(&thp[i]);
    }
    // Programmatic dependent launch: everything above reads only plan tables, which were complete before the
    // previous kernel in the stream passed this same point, so it may run while that kernel drains.  From here
    // on the previous kernel's results are needed; our successor may start its own prologue right away.
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    __syncthreads();

    if (threadIdx.x >= K::GROUPS * K::GT) {
        // ================================ producer warp (one lane) ================================
        // the producer warpgroup hands its registers to the consumers (the CTA pool is 640 x 96: 512 x 112 + 128 x 24)
        if constexpr (CWO_SETMAXNREG) asm volatile("setmaxnreg.dec.sync.aligned.u32 24;");
        if (threadIdx.x != K::GROUPS * K::GT) return;
        const int wc = 1 << P.logwc;
        const int groups = N >> P.logwc, bg = groups < 256 ? groups : 256;    // column groups per TMA box
        auto load = [&](int j) {
            const int b = j % K::NBUF;
            const int gt = blockIdx.x + j * gridDim.x;
            const int plane = batched ? gt / P.tiles_per_plane : 0;
            const int tile = gt - plane * P.tiles_per_plane;
            const float2* in = P.in + (size_t)plane * P.in_plane_stride;
            unsigned char* dst = smraw + b * K::BUF;
            if constexpr (KIND == ROW_FWD) {               // W rows of the row-major field, NP points each
                mbar_expect_tx(&full[b], W * NP * 8);
#pragma unroll
                for (int r = 0; r < W; ++r)
                    bulk_g2s(dst + (size_t)r * RS * 8, in + (size_t)(tile * W + r) * P.pitch, NP * 8, &full[b]);
            } else if constexpr (KIND == ROW_INV) {        // W rows of the column-tiled workspace: [x/Wc][row][x%Wc]
                mbar_expect_tx(&full[b], W * N * 8);
                for (int c = 0; c < groups; c += bg)
                    tma_load_2d(dst + (size_t)c * W * wc * 8, &P.tmap, tile * W * wc * 2, plane * groups + c, &full[b]);
            } else {                                       // column tile: one contiguous [ly][W] block
                const uint32_t bytes = (uint32_t)P.ly * W * 8;
                mbar_expect_tx(&full[b], bytes);
                const unsigned char* src = reinterpret_cast<const unsigned char*>(in + (size_t)tile * P.ly * W);
                constexpr uint32_t CH = 16384;
                for (uint32_t o = 0; o < bytes; o += CH) bulk_g2s(dst + o, src + o, bytes - o < CH ? bytes - o : CH, &full[b]);
            }
        };
        auto store = [&](int j) {
            const int b = j % K::NBUF;
            const int gt = blockIdx.x + j * gridDim.x;
            const int plane = batched ? gt / P.tiles_per_plane : 0;
            const int tile = gt - plane * P.tiles_per_plane;
            float2* out = P.out + (size_t)plane * P.out_plane_stride;
            unsigned char* src = smraw + b * K::BUF;
            if constexpr (KIND == ROW_FWD) {
                for (int c = 0; c < groups; c += bg)
                    tma_store_2d(&P.tmap, src + (size_t)c * W * wc * 8, tile * W * wc * 2, plane * groups + c);
            } else if constexpr (KIND == ROW_INV && IOM == OUT_INTENSITY) {   // W rows of floats, NP points each
                float* outf = reinterpret_cast<float*>(out);
#pragma unroll
                for (int r = 0; r < W; ++r)
                    bulk_s2g(outf + (size_t)(tile * W + r) * P.pitch, src + (size_t)r * RS * 8, NP * 4);
            } else if constexpr (KIND == ROW_INV) {        // W rows of the row-major field, NP points each
#pragma unroll
                for (int r = 0; r < W; ++r)
                    bulk_s2g(out + (size_t)(tile * W + r) * P.pitch, src + (size_t)r * RS * 8, NP * 8);
            } else {
                const uint32_t bytes = (uint32_t)P.ly * W * 8;
                unsigned char* dst = reinterpret_cast<unsigned char*>(out + (size_t)tile * P.ly * W);
                constexpr uint32_t CH = 16384;
                for (uint32_t o = 0; o < bytes; o += CH) bulk_s2g(dst + o, src + o, bytes - o < CH ? bytes - o : CH);
            }
            bulk_commit();
        };
        for (int j = 0; j < nt && j < K::NBUF; ++j) load(j);
        for (int j = 0; j < nt; ++j) {
            mbar_wait_backoff(&staged[j % K::NBUF], (j / K::NBUF) & 1);
            store(j);
            if (j + K::NBUF < nt) {
                bulk_wait_read();                          // the stores have read the buffer
                load(j + K::NBUF);
            }
        }
        asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
        return;
    }

    // ===================================== consumer groups =====================================
    if constexpr (CWO_SETMAXNREG) asm volatile("setmaxnreg.inc.sync.aligned.u32 112;");
    const int g = threadIdx.x >> 8, t = threadIdx.x & 255;
    const SyncGroup sync{1 + g};
    const int us = t / (W / 2), w0 = 2 * (t % (W / 2));     // standard mapping: unit us, lanes w0, w0+1
    const int u[2] = {us, us};
    const int xw = t % W, xi2 = 2 * (t / W);                // unit-pair mapping: lane xw, units xi2, xi2+1

    constexpr bool COLPASS = (KIND != ROW_FWD && KIND != ROW_INV);
#pragma unroll 1
    for (int j = g; j < nt; j += K::GROUPS) {
        const int b = j % K::NBUF;
        const int gt = blockIdx.x + j * gridDim.x;
        const int plane = batched ? gt / P.tiles_per_plane : 0;
        const int tile = gt - plane * P.tiles_per_plane;
        float2* sm = reinterpret_cast<float2*>(smraw + b * K::BUF);
        mbar_wait(&full[b], (j / K::NBUF) & 1);

        if constexpr (COLPASS) {
            // ---- column passes: packed arithmetic, both slots in lockstep (fft_packed.cuh) ----------------
            PV pv;
#pragma unroll
            for (int e = 0; e < 16; ++e) {
                if (e < NE) {
                    const ulonglong2 t2 = *reinterpret_cast<const ulonglong2*>(&sm[(us + e * Q) * W + w0]);
                    pv.r[e] = t2.x; pv.i[e] = t2.y;                    // the workspace stores lane pairs planar
                } else {
                    pv.r[e] = pv.i[e] = 0ull;
                }
            }
            typename PipeMidSelect<LOGN, KIND == COL_FWD ? MID_NONE : MID>::type mid(P, u, tile * W + w0, batched ? nullptr : thy, plane);
            if constexpr (KIND == COL_FWD) {
                transform_p<LOGN, true, false, false>(pv, us, w0, sm, tws, mid, sync);
            } else if constexpr (KIND == COL_FUSED) {
                transform_p<LOGN, true, true, false>(pv, us, w0, sm, tws, mid, sync);
            } else {
                transform_p<LOGN, false, true, true>(pv, us, w0, sm, tws, mid, sync);
            }
            sync();                                           // nobody still reads the exchange image
            // inverse column results stay conjugated: pass R' expects conj(field)
#pragma unroll
            for (int e = 0; e < NE; ++e) {
                *reinterpret_cast<ulonglong2*>(&sm[(us + e * Q) * W + w0]) = make_ulonglong2(pv.r[e], pv.i[e]);
            }
            fence_proxy_async();
            mbar_arrive(&staged[b]);
            continue;
        }
        static_assert(COLPASS || KIND == ROW_FWD || KIND == ROW_INV, "kind");
        if constexpr (!PAD) {
            // ---- unpadded row passes: packed arithmetic on (even bins, odd bins) lane pairs ------------------------
            // One radix-2 step splits a row of n = 2h points into two h-point lanes with the same twiddles
            // (rowfft scheme: forward a = x[m] + x[m+h], b = (x[m] - x[m+h]) w^m, X[2j] = FFT_h(a)[j], X[2j+1] =
            // FFT_h(b)[j]; inverse x[m] = A[m] + w^-m B[m], x[m+h] = A[m] - w^-m B[m]).  (X[2j], X[2j+1]) is one planar
            // 16-byte element of the column-tiled workspace = the register pair: half the butterfly instructions of
            // the scalar form, no unit-pair mapping.  The tile's W rows are the W lane pairs of Tile<LOGN-1>.
            using CH = Tile<LOGN - 1>;
            static_assert(CH::T == K::GT && CH::W == 2 * W && CH::SMEM_BYTES <= K::BUF, "half-length tile shape");
            constexpr int QH = CH::Q, H = CH::N;
            const int hus = t / W, hr = t % W;                // unit and row of this thread
            const float2 wb = tws[hus];                       // w^us (n-point table); w^(us + e QH) = wb w32^e
            float2 tq[8];
#pragma unroll
            for (int e = 0; e < 8; ++e) tq[e] = e == 0 ? wb : cmul(wb, w32_pow(e));
            PV pv;
            if constexpr (KIND == ROW_FWD) {
                const float2* x = sm + hr * RS + hus;
#pragma unroll
                for (int e = 0; e < 16; ++e) {
                    const float2 lo = x[e * QH], hi = x[H + e * QH];
                    const float2 a = cadd(lo, hi), d = csub(lo, hi);
                    const float2 bb = e < 8 ? cmul(d, tq[e]) : cmul_mi(cmul(d, tq[e - 8]));
                    pv.r[e] = pk_make(a.x, bb.x); pv.i[e] = pk_make(a.y, bb.y);
                }
                sync();                                       // staged image retired: the buffer is the exchange buffer now
                transform_p<LOGN - 1, true, false, false>(pv, hus, 2 * hr, sm, twh, MidNone(), sync);
                sync();                                       // nobody still reads the exchange image
                // [x/Wc][row][x%Wc]: the pair (2j, 2j+1), j = hus + e QH, of row hr
#pragma unroll
                for (int e = 0; e < 16; ++e) {
                    const int x2 = 2 * (hus + e * QH);
                    float2* d = sm + ((((x2 >> P.logwc) * W + hr) << P.logwc) + (x2 & ((1 << P.logwc) - 1)));
                    *reinterpret_cast<ulonglong2*>(d) = make_ulonglong2(pv.r[e], pv.i[e]);
                }
            } else {
#pragma unroll
                for (int e = 0; e < 16; ++e) {
                    const int x2 = 2 * (hus + e * QH);
                    const float2* d = sm + ((((x2 >> P.logwc) * W + hr) << P.logwc) + (x2 & ((1 << P.logwc) - 1)));
                    const ulonglong2 q2 = *reinterpret_cast<const ulonglong2*>(d);
                    pv.r[e] = q2.x; pv.i[e] = q2.y;           // conj(field): see the column store
                }
                sync();                                       // staged image retired
                transform_p<LOGN - 1, false, true, false>(pv, hus, 2 * hr, sm, twh, MidNone(), sync);
                sync();                                       // nobody still reads the exchange image
                const float sc = P.out_scale;                 // conj completes the inverse transform
                if constexpr (IOM == OUT_INTENSITY) {
                    float* y = reinterpret_cast<float*>(sm) + hr * RS * 2 + hus;
#pragma unroll
                    for (int e = 0; e < 16; ++e) {
                        float ar, br, ai, bi;
                        pk_split(pv.r[e], ar, br); pk_split(pv.i[e], ai, bi);
                        const float2 m = cmul(make_float2(br, bi), e < 8 ? tq[e] : cmul_mi(tq[e - 8]));
                        const float2 lo = make_float2(ar + m.x, ai + m.y), hi = make_float2(ar - m.x, ai - m.y);
                        if (P.real_mode == REAL_ABS2) {
                            y[e * QH] = (lo.x * lo.x + lo.y * lo.y) * (sc * sc);
                            y[H + e * QH] = (hi.x * hi.x + hi.y * hi.y) * (sc * sc);
                        } else {
                            y[e * QH] = real_field(lo.x, lo.y, sc, P.real_mode);
                            y[H + e * QH] = real_field(hi.x, hi.y, sc, P.real_mode);
                        }
                    }
                } else if constexpr (IOM == OUT_PHASOR_AMP) {
                    // GS constraints (S10; Listing 8 lines 11-13 / 15-16): keep u/|u| (1 where u == 0), impose the amplitude
                    // of the next plane.  The amplitudes of all the thread's samples are requested before the first is used.
                    const float* am = P.out_amp + (size_t)(tile * W + hr) * P.pitch + hus;
                    float alo[16], ahi[16];
#pragma unroll
                    for (int e = 0; e < 16; ++e) { alo[e] = __ldg(&am[e * QH]); ahi[e] = __ldg(&am[H + e * QH]); }
                    float2* y = sm + hr * RS + hus;
                    auto constrain = [](float2 u, float a) {           // u is conj(sample)
                        const float m2 = u.x * u.x + u.y * u.y;
                        float2 ph = make_float2(1.f, 0.f);
                        if (m2 > 0.f) { const float r = rsqrtf(m2); ph = make_float2(u.x * r, -u.y * r); }
                        return make_float2(a * ph.x, a * ph.y);
                    };
#pragma unroll
                    for (int e = 0; e < 16; ++e) {
                        float ar, br, ai, bi;
                        pk_split(pv.r[e], ar, br); pk_split(pv.i[e], ai, bi);
                        const float2 m = cmul(make_float2(br, bi), e < 8 ? tq[e] : cmul_mi(tq[e - 8]));
                        y[e * QH] = constrain(make_float2(ar + m.x, ai + m.y), alo[e]);
                        y[H + e * QH] = constrain(make_float2(ar - m.x, ai - m.y), ahi[e]);
                    }
                } else {
                    float2* y = sm + hr * RS + hus;
#pragma unroll
                    for (int e = 0; e < 16; ++e) {
                        float ar, br, ai, bi;
                        pk_split(pv.r[e], ar, br); pk_split(pv.i[e], ai, bi);
                        const float2 m = cmul(make_float2(br, bi), e < 8 ? tq[e] : cmul_mi(tq[e - 8]));
                        y[e * QH] = make_float2((ar + m.x) * sc, -(ai + m.y) * sc);
                        y[H + e * QH] = make_float2((ar - m.x) * sc, -(ai - m.y) * sc);
                    }
                }
            }
            fence_proxy_async();
            mbar_arrive(&staged[b]);
            continue;
        }
        // ---- padded row passes: scalar arithmetic, the two slots half a stage apart (pp_core.cuh) --------
        float2 v[2][16];

        // ---- registers <- staged tile ------------------------------------------------------------
        if constexpr (KIND == ROW_FWD) {
#pragma unroll
            for (int s = 0; s < 2; ++s)
#pragma unroll
                for (int e = 0; e < 16; ++e)
                    v[s][e] = (e < NE) ? sm[(w0 + s) * RS + us + e * Q] : make_float2(0.f, 0.f);
        } else if constexpr (KIND == ROW_INV) {
            // [x/Wc][row][x%Wc]: points (x, x+1) of row xw, x = xi2 + e*Q, are 16 bytes
            const float2* src = sm + ((((xi2 >> P.logwc) * W + xw) << P.logwc) + (xi2 & ((1 << P.logwc) - 1)));
#pragma unroll
            for (int e = 0; e < 16; ++e) {
                const float4 t4 = *reinterpret_cast<const float4*>(src + e * Q * W);
                v[0][e] = make_float2(t4.x, t4.z); v[1][e] = make_float2(t4.y, t4.w);   // planar pair; conj(field): see the column store
            }
        }

        // ---- transform: ping-pong schedule of pp_core.cuh ----------------------------------------------
        constexpr int M = C::M, L0 = C::L0;
        float2* rgA = sm;
        float2* rgB = sm + PP<LOGN>::REGION;
        const int wh = w0 >> 1;
        if constexpr (KIND == ROW_FWD) {
            sync();                                           // staged image retired
            pp_run<LOGN, true, 0, M - 1, false>(v, us, wh, rgA, rgB, tws, sync);
            // stage M-2 -> one plane per lane, read back unit pairs, last stage in unit-pair mapping
            constexpr int lns = L0 + 4 * (M - 2);
            sync();
            {
                const int j0 = ((us >> lns) << (lns + 4)) + (us & ((1 << lns) - 1));
                float2* pl = sm + w0 * C::XPLANE;
#pragma unroll
                for (int q = 0; q < 16; ++q) {
                    const int p = j0 + (q << lns), pi = p + 2 * (p >> 4);
                    pl[pi] = v[0][perm<16>(q)];
                    pl[C::XPLANE + pi] = v[1][perm<16>(q)];
                }
            }
            sync();
#pragma unroll
            for (int e = 0; e < 16; ++e) {
                const int p = xi2 + e * Q;
                const float4 x = *reinterpret_cast<const float4*>(&sm[xw * C::XPLANE + p + 2 * (p >> 4)]);
                v[0][e] = make_float2(x.x, x.y);
                v[1][e] = make_float2(x.z, x.w);
            }
            const int ux[2] = {xi2, xi2 + 1};
            butterflies<LOGN, 4, true, true>(v, ux, L0 + 4 * (M - 1), tws);
            unpermute<16>(v[0]); unpermute<16>(v[1]);
        } else if constexpr (KIND == ROW_INV) {
            dft16(v[0]); dft16(v[1]);                         // unit-pair mapping, Ns = 1: no twiddles
            sync();
            {
                float2* rg = (xw & 1) ? rgB : rgA;
#pragma unroll
                for (int s = 0; s < 2; ++s)
#pragma unroll
                    for (int q = 0; q < 16; ++q) rg[ridx<LOGN>(16 * (xi2 + s) + q, xw >> 1)] = v[s][perm<16>(q)];
            }
            sync();
            lds_slot<LOGN>(v[0], us, wh, rgA);
            lds_slot<LOGN>(v[1], us, wh, rgB);
            sync();                                           // regions free again for pp_run
            pp_run<LOGN, false, M + 1, 2 * M, true>(v, us, wh, rgA, rgB, tws, sync);
            if constexpr (L0 == 0) { unpermute<16>(v[0]); unpermute<16>(v[1]); }
        }

        // ---- results -> the same buffer, in the layout of the destination; the producer stores them ----
        sync();                                               // nobody still reads the exchange regions
        if constexpr (KIND == ROW_FWD) {
            // [x/Wc][row][x%Wc]; register e of slot s <-> point xi2 + s + e*Q of row xw
            float2* d = sm + ((((xi2 >> P.logwc) * W + xw) << P.logwc) + (xi2 & ((1 << P.logwc) - 1)));
#pragma unroll
            for (int e = 0; e < 16; ++e)
                *reinterpret_cast<float4*>(d + e * Q * W) = make_float4(v[0][e].x, v[1][e].x, v[0][e].y, v[1][e].y);
        } else if constexpr (KIND == ROW_INV) {
            static_assert(!PAD || IOM == OUT_COMPLEX || IOM == OUT_INTENSITY, "padded rows: GS store modes run in pass_kernel");
            const float sc = P.out_scale;                     // conj completes the inverse transform
            if constexpr (IOM == OUT_INTENSITY) {             // Eq.(20): |u|^2 as floats, same row stride (bytes) of the staging
                float* smf = reinterpret_cast<float*>(sm);
#pragma unroll
                for (int s = 0; s < 2; ++s)
#pragma unroll
                    for (int e = 0; e < NE; ++e)
                        smf[(w0 + s) * RS * 2 + us + e * Q] =
                            P.real_mode == REAL_ABS2 ? (v[s][e].x * v[s][e].x + v[s][e].y * v[s][e].y) * (sc * sc)
                                                     : real_field(v[s][e].x, v[s][e].y, sc, P.real_mode);
            } else {
#pragma unroll
                for (int s = 0; s < 2; ++s)
#pragma unroll
                    for (int e = 0; e < NE; ++e)
                        sm[(w0 + s) * RS + us + e * Q] = make_float2(v[s][e].x * sc, -v[s][e].y * sc);
            }
        }
        fence_proxy_async();
        mbar_arrive(&staged[b]);
    }
}

template <int LOGN, int KIND, bool PAD, int MID, int IOM>
static cudaError_t launch_pipe(int n_tiles, cudaStream_t s, const PassParams& p) {
    using K = PipeCfg<LOGN, KIND>;
    constexpr size_t SM = (MID == MID_ASM_SPLIT) ? K::SMEM_TAB : K::SMEM_NOTAB;
    DeviceInfo* d = device_info();
    if (!d) return cudaErrorInvalidDevice;
    const int n_sm = d->n_sm;
    static FuncOnce once;
    if (!once.done(d->index)) {
        cudaError_t e = cudaFuncSetAttribute(pipe_kernel<LOGN, KIND, PAD, MID, IOM>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SM);
        if (e != cudaSuccess) return e;
        once.set(d->index);
    }
    PassParams q = p;
    q.n_tiles = n_tiles;
    const int grid = n_tiles < n_sm ? n_tiles : n_sm;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3((unsigned)K::THREADS);
    cfg.dynamicSmemBytes = SM; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, pipe_kernel<LOGN, KIND, PAD, MID, IOM>, q);
}

}  // namespace cwo
