// pass_kernel.cuh -- one streaming pass over the field: every CTA loads a tile of W lanes x n points,
// transforms it on chip and stores it.  The passes of a propagation:
//   ROW_FWD     rows of u1 (row-major)  -> FFT_x  -> workspace in column-tile order      (pass R)
//   COL_FUSED   column tile of the workspace -> FFT_y -> x H -> IFFT_y -> same tile        (pass C)
//   ROW_INV     rows of the workspace   -> IFFT_x -> u2 (row-major)                        (pass R')
//   COL_FWD / COL_MIDINV   the two halves of pass C, for the depth stack (S9)
// PAD (Fresnel): the transform length is twice the number of stored points; the zero half is never
// loaded (S3) and the discarded half never stored (S8) -- the compiler prunes the butterflies that
// only see zeros / only feed discarded outputs.  GS constraints (S10) are load/store modes of the
// row passes.  H (S2) is produced in registers by the Mid functors.
//
// Workspace layout ("column-tile order"): T[x / Wc][y][x % Wc], y < Ny, Wc = lanes of the column
// pass; a column pass reads and writes one contiguous Ny*Wc block.  For Wc >= 2 two neighbouring
// columns (x even, x + 1) share one 16-byte element stored PLANAR, (re_x, re_x+1, im_x, im_x+1): that is
// the register-pair format of the packed arithmetic (fft_packed.cuh), so no pass ever shuffles registers
// to (de)interleave.  Wc == 1 (n = 16384) keeps interleaved (re, im).
#pragma once
#ifndef CWO_SPLIT_SYNC
#define CWO_SPLIT_SYNC 1
#endif
#include "cwo_internal.h"
#include "fft_core.cuh"
#include "pp_core.cuh"
#include "fft_packed.cuh"

namespace cwo {

enum { ROW_FWD = 0, ROW_INV = 1, COL_FWD = 2, COL_FUSED = 3, COL_MIDINV = 4 };

// element (x = p, y = row) of the column-tiled workspace, any tile width (generic, 32-bit accesses when planar)
__device__ __forceinline__ size_t ws_block(int p, int row, int ly, int logwc) {
    return ((size_t)(p >> logwc) * ly + row) << logwc;                         // complex elements
}
__device__ __forceinline__ float2 ws_load(const float2* ws, int p, int row, int ly, int logwc) {
    const int c = p & ((1 << logwc) - 1);
    if (logwc == 0) return ws[ws_block(p, row, ly, 0)];
    const float* f = reinterpret_cast<const float*>(ws + ws_block(p, row, ly, logwc)) + ((c >> 1) << 2) + (c & 1);
    return make_float2(f[0], f[2]);
}
__device__ __forceinline__ void ws_store(float2* ws, int p, int row, int ly, int logwc, float2 v) {
    const int c = p & ((1 << logwc) - 1);
    if (logwc == 0) { ws[ws_block(p, row, ly, 0)] = v; return; }
    float* f = reinterpret_cast<float*>(ws + ws_block(p, row, ly, logwc)) + ((c >> 1) << 2) + (c & 1);
    f[0] = v.x; f[2] = v.y;
}

struct MidNone {
    __device__ __forceinline__ void operator()(float2 (&)[2][16]) const {}
    __device__ __forceinline__ void packed(PV&) const {}
};

// Fresnel: FFT2 of the sampled separable chirp is the outer product Cx[k]*Cy[l] (S2, S7 folded in)
template <int LOGN> struct MidTables {
    const PassParams& P; const int (&u)[2]; int lane0; float2* sm;
    __device__ __forceinline__ void operator()(float2 (&v)[2][16]) const {
        using C = Tile<LOGN>;
        const float2 cx0 = __ldg(&P.tab_lane[lane0]);
        const float2 cx1 = __ldg(&P.tab_lane[C::PAIR ? lane0 + 1 : lane0]);
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            const float2 cy0 = __ldg(&P.tab_point[u[0] + e * C::Q]);
            const float2 cy1 = C::PAIR ? cy0 : __ldg(&P.tab_point[u[1] + e * C::Q]);
            v[0][e] = cconj(cmul(v[0][e], cmul(cx0, cy0)));
            v[1][e] = cconj(cmul(v[1][e], cmul(cx1, cy1)));
        }
    }
    // both slots in packed form (fft_packed.cuh); lane pairs only
    __device__ __forceinline__ void packed(PV& v) const {
        using C = Tile<LOGN>;
        const float2 cx0 = __ldg(&P.tab_lane[lane0]), cx1 = __ldg(&P.tab_lane[lane0 + 1]);
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            const float2 cy = __ldg(&P.tab_point[u[0] + e * C::Q]);
            float r0, r1, i0, i1;
            pk_split(v.r[e], r0, r1); pk_split(v.i[e], i0, i1);
            const float2 a = cmul(make_float2(r0, i0), cmul(cx0, cy)), b = cmul(make_float2(r1, i1), cmul(cx1, cy));
            v.r[e] = pk_make(a.x, b.x); v.i[e] = pk_make(-a.y, -b.y);
        }
    }
};

// ASM, Eq.(16), phase in cycles = z/lambda - ax k^2 - ay l^2 - res(k,l):
// constant + paraxial parts from fp64-built 1-D tables (theta_lane includes z/lambda), the small
// non-paraxial residual res = (z/lambda) s^2 / (2 (1+sqrt(1-s))^2), s = lambda^2 (fx^2+fy^2), in fp32
// (no cancellation).  Only used when the plan has verified that no bin is evanescent and res is small.
template <int LOGN> struct MidAsmSplit {
    const PassParams& P; const int (&u)[2]; int lane0; float2* sm;
    __device__ __forceinline__ void operator()(float2 (&v)[2][16]) const {
        using C = Tile<LOGN>;
        const float* thl = reinterpret_cast<const float*>(P.tab_lane);
        const float* thp = reinterpret_cast<const float*>(P.tab_point);
        float thx[2], sx[2];
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            const int lane = lane0 + (C::PAIR ? s : 0);
            const int ks = (lane < P.n_lane_bins / 2) ? lane : lane - P.n_lane_bins;
            thx[s] = __ldg(&thl[lane]);
            sx[s] = P.res_a * (float)ks * (float)ks;
        }
#pragma unroll
        for (int e = 0; e < 16; ++e) {
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                const int l = u[C::PAIR ? 0 : s] + e * C::Q;
                const int ls = (l < C::N / 2) ? l : l - C::N;
                const float sv = fmaf(P.res_b * (float)ls, (float)ls, sx[s]);
                const float om = 1.0f - sv;
                const float r = 1.0f + om * rsqrtf(om);
                const float res = __fdividef(P.res_c * sv * sv, 2.0f * r * r);
                float ph = thx[s] + __ldg(&thp[l]) - res;
                ph -= rintf(ph);
                float sn, cs;
                __sincosf(6.283185307179586f * ph, &sn, &cs);
                v[s][e] = cconj(cmul(v[s][e], make_float2(cs, sn)));
                if (P.band) {                              // Eq.(18): the two Rect band limits
                    const int lane = lane0 + (C::PAIR ? s : 0);
                    const int ks = (lane < P.n_lane_bins / 2) ? lane : lane - P.n_lane_bins;
                    if (ks < P.band_lane_lo || ks > P.band_lane_hi || ls < P.band_point_lo || ls > P.band_point_hi)
                        v[s][e] = make_float2(0.f, 0.f);
                }
            }
        }
    }
};

// ASM with the phase evaluated in fp64 per sample (general path: evanescent bins, long distances).
// w = 1/lambda^2 - (fx^2 + fy^2) uses the oracle's expression and rounding for the evanescent test.
// H is staged through the (idle) tile buffer by a rolled loop to keep the code small.
template <int LOGN> struct MidAsmF64 {
    const PassParams& P; const int (&u)[2]; int lane0; float2* sm;
    __device__ __forceinline__ void operator()(float2 (&v)[2][16]) const {
        using C = Tile<LOGN>;
        __syncthreads();                                   // tile buffer no longer being read
        float2* mine = sm + threadIdx.x;
#pragma unroll 1
        for (int i = 0; i < 32; ++i) {
            const int s = i & 1, e = i >> 1;
            const int lane = lane0 + (C::PAIR ? s : 0);
            const int l = u[C::PAIR ? 0 : s] + e * C::Q;
            const int ks = (lane < P.n_lane_bins / 2) ? lane : lane - P.n_lane_bins;
            const int ls = (l < C::N / 2) ? l : l - C::N;
            const double fx = (double)ks * P.df_lane, fy = (double)ls * P.df_point;
            const double w = __dsub_rn(P.inv_lam2, __dadd_rn(__dmul_rn(fx, fx), __dmul_rn(fy, fy)));
            float2 m = make_float2(0.f, 0.f);
            const bool cut = P.band && (ks < P.band_lane_lo || ks > P.band_lane_hi || ls < P.band_point_lo ||
                                        ls > P.band_point_hi);
            if (w >= 0.0 && !cut) {
                double c = P.z * sqrt(w) + (P.off_lane * fx + P.off_point * fy);
                c -= rint(c);
                float sn, cs;
                sincospif(2.0f * (float)c, &sn, &cs);
                m = make_float2(cs, sn);
            }
            mine[i * C::T] = m;
        }
#pragma unroll
        for (int e = 0; e < 16; ++e)
#pragma unroll
            for (int s = 0; s < 2; ++s) v[s][e] = cconj(cmul(v[s][e], mine[(2 * e + s) * C::T]));
    }
};

template <int LOGN, int MID> struct MidSelect;
template <int LOGN> struct MidSelect<LOGN, MID_TABLES> { using type = MidTables<LOGN>; };
template <int LOGN> struct MidSelect<LOGN, MID_ASM_SPLIT> { using type = MidAsmSplit<LOGN>; };
template <int LOGN> struct MidSelect<LOGN, MID_ASM_F64> { using type = MidAsmF64<LOGN>; };

// Mid functors with a packed() form (pipe_kernel.cuh); constructor (P, u, lane0, theta_y in shared memory or
// nullptr for the global table, plane)
template <int LOGN, int MID> struct PipeMidSelect;

// IOM: ROW_FWD -> InMode of the load, ROW_INV -> OutMode of the store, column passes -> 0.
// X (row passes over a workspace of 2-wide column tiles, W == 2): unit-pair mapping at the workspace side.
template <int LOGN, int KIND, bool PAD, int MID, int IOM, bool X>
__global__ void __launch_bounds__(Tile<LOGN>::T, Tile<LOGN>::MINB)
pass_kernel(const __grid_constant__ PassParams P) {
    using C = Tile<LOGN>;
    constexpr int W = C::W, Q = C::Q;
    constexpr bool ROWPASS = (KIND == ROW_FWD || KIND == ROW_INV);
    constexpr int NE = PAD ? 8 : 16;        // PAD: points >= n/2 are zero on load / dropped on store
    extern __shared__ float2 sm[];
    // launched with programmatic stream serialization: resident as soon as the previous kernel's CTAs leave,
    // running once its results are complete
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

    const int tile = blockIdx.x;
    int u[2], w0;
    if constexpr (C::PAIR) {
        w0 = 2 * (threadIdx.x % (W / 2));
        u[0] = u[1] = threadIdx.x / (W / 2);
    } else {
        w0 = 0;
        u[0] = threadIdx.x; u[1] = threadIdx.x + Q / 2;
    }
    const int lane0 = tile * W + w0;        // row (row pass) or column (column pass) of slot 0
    if constexpr (!ROWPASS && C::PAIR && MID != MID_ASM_F64 && LOGN >= 8) {
        // column passes on lane pairs: packed f32x2 arithmetic, both slots in lockstep (fft_packed.cuh); the
        // workspace stores the pair planar, which is the register format
        const ulonglong2* src = reinterpret_cast<const ulonglong2*>(P.in + (size_t)tile * P.ly * W);
        ulonglong2* dst = reinterpret_cast<ulonglong2*>(P.out + (size_t)tile * P.ly * W);
        // the tile of the CTA that will take this one's place on the SM: have L2 fetch it now, so that its loads
        // (nothing overlaps them: the whole tile goes to registers before the first butterfly) find it on chip
        if (threadIdx.x == 0 && P.pf_dist > 0 && tile + P.pf_dist < P.n_tiles)
            l2_prefetch(P.in + (size_t)(tile + P.pf_dist) * P.ly * W, (uint32_t)(P.ly * W * 8));
        // stage twiddles: copied to shared memory behind the exchange buffer (the first stage has none, so the copy is
        // covered by it); read from global memory they are evicted from L1 by the tile traffic and every stage
        // would begin with an L2 round trip
        float2* tws = reinterpret_cast<float2*>(reinterpret_cast<unsigned char*>(sm) + C::SMEM_BYTES + 64);
        for (int i = threadIdx.x; i < PP<LOGN>::NTW_P; i += C::T) tws[i] = __ldg(&P.tw[i]);
        PV pv;
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            if (e < NE) {
                const ulonglong2 t2 = __ldcs(&src[((size_t)(u[0] + e * Q) * W + w0) >> 1]);   // streamed: keep L1 for the tables
                pv.r[e] = t2.x; pv.i[e] = t2.y;
            } else {
                pv.r[e] = pv.i[e] = 0ull;
            }
        }
        typename PipeMidSelect<LOGN, KIND == COL_FWD ? MID_NONE : MID>::type mid(P, u, lane0, nullptr, 0);
#if CWO_SPLIT_SYNC
        // split-phase exchange synchronisation on two mbarriers behind the tile buffer (fft_core.cuh SyncSplit)
        uint64_t* bars = reinterpret_cast<uint64_t*>(reinterpret_cast<unsigned char*>(sm) + C::SMEM_BYTES);
        if (threadIdx.x == 0) {
            mbar_init(&bars[0], C::T); mbar_init(&bars[1], C::T);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
        __syncthreads();
        const SyncSplit sy{&bars[0], &bars[1], 0u, 0u};
        sy.consumed();                                     // the region starts free
#else
        __syncthreads();
        const SyncCta sy;
#endif
        if constexpr (KIND == COL_FWD) transform_p<LOGN, true, false, false>(pv, u[0], w0, sm, tws, mid, sy);
        else if constexpr (KIND == COL_FUSED) transform_p<LOGN, true, true, false>(pv, u[0], w0, sm, tws, mid, sy);
        else transform_p<LOGN, false, true, true>(pv, u[0], w0, sm, tws, mid, sy);
#pragma unroll
        for (int e = 0; e < NE; ++e) __stcs(&dst[((size_t)(u[0] + e * Q) * W + w0) >> 1], make_ulonglong2(pv.r[e], pv.i[e]));
        return;
    }
    float2 v[2][16];

    // ---- load -----------------------------------------------------------------------------------
    if constexpr (KIND == ROW_FWD) {
        // rows of a row-major field; slot s = row lane0 + s (PAIR) / same row, second unit (!PAIR)
        if constexpr (IOM == IN_COMPLEX) {
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                const int row = lane0 + (C::PAIR ? s : 0);
                const bool ok = row < P.rows;
                const size_t base = (size_t)row * P.pitch + u[s];
#pragma unroll
                for (int e = 0; e < 16; ++e)
                    v[s][e] = (e < NE && ok) ? P.in[base + e * Q] : make_float2(0.f, 0.f);
            }
        } else {
            // GS step 1: amp * exp(i phase) (Listing 8 lines 3-5).  Accurate sincosf is bulky, so the
            // samples are formed by a rolled loop and staged through the thread's own slots of the
            // (still idle) tile buffer.
            float2* mine = sm + threadIdx.x;
#pragma unroll 1
            for (int i = 0; i < 2 * NE; ++i) {
                const int s = i & 1, e = i >> 1;
                const int row = lane0 + (C::PAIR ? s : 0);
                float2 x = make_float2(0.f, 0.f);
                if (row < P.rows) {
                    const size_t a = (size_t)row * P.pitch + (s ? u[1] : u[0]) + e * Q;
                    float sn, cs;
                    sincosf(P.in_phase[a], &sn, &cs);
                    const float am = P.in_amp[a];
                    x = make_float2(am * cs, am * sn);
                }
                mine[i * C::T] = x;
            }
#pragma unroll
            for (int s = 0; s < 2; ++s)
#pragma unroll
                for (int e = 0; e < 16; ++e) v[s][e] = (e < NE) ? mine[(2 * e + s) * C::T] : make_float2(0.f, 0.f);
        }
    } else if constexpr (KIND == ROW_INV && X) {
        // rows of the column-tiled workspace, 2-wide tiles: points (x, x+1) of row tile*2 + w are 16 bytes
        const int row = tile * 2 + (threadIdx.x & 1);
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            const int x = (threadIdx.x & ~1) + e * Q;
            const float4 t4 = *reinterpret_cast<const float4*>(&P.in[((size_t)(x >> 1) * P.ly + row) * 2]);
            v[0][e] = make_float2(t4.x, t4.z); v[1][e] = make_float2(t4.y, t4.w);
        }
    } else if constexpr (KIND == ROW_INV) {
        // rows of the column-tiled workspace
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            const int row = lane0 + (C::PAIR ? s : 0);
            const bool ok = row < P.rows;
#pragma unroll
            for (int e = 0; e < 16; ++e) {
                v[s][e] = ok ? ws_load(P.in, u[s] + e * Q, row, P.ly, P.logwc) : make_float2(0.f, 0.f);
            }
        }
    } else {
        // column tile: contiguous [ly][W] block; a PAIR thread reads both lanes with one 128-bit load
        const float2* src = P.in + (size_t)tile * P.ly * W;
        if constexpr (C::PAIR) {
#pragma unroll
            for (int e = 0; e < 16; ++e) {
                if (e < NE) {
                    const float4 t = *reinterpret_cast<const float4*>(&src[(size_t)(u[0] + e * Q) * W + w0]);
                    v[0][e] = make_float2(t.x, t.z); v[1][e] = make_float2(t.y, t.w);
                } else {
                    v[0][e] = v[1][e] = make_float2(0.f, 0.f);
                }
            }
        } else {
#pragma unroll
            for (int s = 0; s < 2; ++s)
#pragma unroll
                for (int e = 0; e < 16; ++e)
                    v[s][e] = (!PAD || u[s] + e * Q < C::N / 2) ? src[u[s] + e * Q] : make_float2(0.f, 0.f);
        }
    }

    // ---- transform ------------------------------------------------------------------------------
    if constexpr (KIND == ROW_FWD && X) {
        transform_fwd_xlast<LOGN>(v, threadIdx.x, sm, P.tw, SyncCta());
    } else if constexpr (KIND == ROW_INV && X) {
        transform_inv_xfirst<LOGN>(v, threadIdx.x, sm, P.tw, SyncCta());
    } else if constexpr (KIND == ROW_FWD || KIND == COL_FWD) {
        transform<LOGN, true, false>(v, u, w0, sm, P.tw, MidNone(), SyncCta());
    } else if constexpr (KIND == ROW_INV) {
        transform<LOGN, false, true>(v, u, w0, sm, P.tw, MidNone(), SyncCta());
    } else {
        typename MidSelect<LOGN, MID>::type mid{P, u, lane0, sm};
        if constexpr (KIND == COL_FUSED) {
            transform<LOGN, true, true>(v, u, w0, sm, P.tw, mid, SyncCta());
        } else {
            mid(v);
            transform<LOGN, false, true>(v, u, w0, sm, P.tw, MidNone(), SyncCta());
        }
    }

    // ---- store (conj completes an inverse transform) -----------------------------------------------
    if constexpr (KIND == ROW_FWD && X) {
        const int row = tile * 2 + (threadIdx.x & 1);
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            const int x = (threadIdx.x & ~1) + e * Q;
            *reinterpret_cast<float4*>(&P.out[((size_t)(x >> 1) * P.ly + row) * 2]) =
                make_float4(v[0][e].x, v[1][e].x, v[0][e].y, v[1][e].y);
        }
    } else if constexpr (KIND == ROW_FWD) {
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            const int row = lane0 + (C::PAIR ? s : 0);
            if (row < P.rows) {
#pragma unroll
                for (int e = 0; e < 16; ++e) {
                    ws_store(P.out, u[s] + e * Q, row, P.ly, P.logwc, v[s][e]);
                }
            }
        }
    } else if constexpr (KIND == ROW_INV) {
        if constexpr (IOM == OUT_COMPLEX) {
            const float sc = P.out_scale;
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                const int row = lane0 + (C::PAIR ? s : 0);
                if (row >= P.rows) continue;
                const size_t base = (size_t)row * P.pitch + u[s];
#pragma unroll
                for (int e = 0; e < NE; ++e) P.out[base + e * Q] = make_float2(v[s][e].x * sc, -v[s][e].y * sc);
            }
        } else if constexpr (IOM == OUT_PHASOR_AMP) {
            // GS constraints (S10), phase constraint then amplitude constraint (Listing 8 lines 11-13 / 15-16): keep
            // u/|u| (1 where u == 0), replace the amplitude by that of the next plane.  The amplitudes of all the
            // thread's samples are requested before the first is used.
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                const int row = lane0 + (C::PAIR ? s : 0);
                if (row >= P.rows) continue;
                const size_t base = (size_t)row * P.pitch + u[s];
                float am[NE];
#pragma unroll
                for (int e = 0; e < NE; ++e) am[e] = P.out_amp[base + e * Q];
#pragma unroll
                for (int e = 0; e < NE; ++e) {
                    const float2 x = v[s][e];                  // the sample is conj(x)
                    const float m2 = x.x * x.x + x.y * x.y;
                    float2 ph = make_float2(1.f, 0.f);
                    if (m2 > 0.f) { const float r = rsqrtf(m2); ph = make_float2(x.x * r, -x.y * r); }
                    P.out[base + e * Q] = make_float2(am[e] * ph.x, am[e] * ph.y);
                }
            }
        } else if constexpr (IOM == OUT_INTENSITY) {
            // Eq.(20): I = |u|^2, one float per sample
            const float sc2 = P.out_scale * P.out_scale;
            float* outf = reinterpret_cast<float*>(P.out);
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                const int row = lane0 + (C::PAIR ? s : 0);
                if (row >= P.rows) continue;
                const size_t base = (size_t)row * P.pitch + u[s];
                if (P.real_mode == REAL_ABS2) {
#pragma unroll
                    for (int e = 0; e < NE; ++e) outf[base + e * Q] = (v[s][e].x * v[s][e].x + v[s][e].y * v[s][e].y) * sc2;
                } else {                                        // |u|, Re u, Im u (section 5); the sample is conj(v)
#pragma unroll
                    for (int e = 0; e < NE; ++e) outf[base + e * Q] = real_field(v[s][e].x, v[s][e].y, P.out_scale, P.real_mode);
                }
            }
        } else {
            // OUT_PHASE, Eq.(25) P:L482 as atan2, by a rolled loop over the thread's samples staged through its own
            // slots of the tile buffer (atan2f would otherwise be unrolled 32 times).
            __syncthreads();                               // tile buffer no longer being read
            float2* mine = sm + threadIdx.x;
#pragma unroll
            for (int s = 0; s < 2; ++s)
#pragma unroll
                for (int e = 0; e < NE; ++e) mine[(2 * e + s) * C::T] = v[s][e];
#pragma unroll 1
            for (int i = 0; i < 2 * NE; ++i) {
                const int s = i & 1, e = i >> 1;
                const int row = lane0 + (C::PAIR ? s : 0);
                if (row >= P.rows) continue;
                const size_t a = (size_t)row * P.pitch + (s ? u[1] : u[0]) + e * Q;
                const float2 x = mine[i * C::T];          // the sample is conj(x)
                // phasor(0) = 1 (cwo.h): an exactly zero sample has phase 0, whatever the signs of its zeros
                reinterpret_cast<float*>(P.out)[a] = (x.x == 0.0f && x.y == 0.0f) ? 0.0f : atan2f(-x.y, x.x);
            }
        }
    } else {
        float2* dst = P.out + (size_t)tile * P.ly * W;
        // An inverse column transform leaves conj(result) here: the conj that would complete it and the conj
        // that opens the inverse row transform of pass R' cancel, so neither is applied.
        constexpr bool CONJ = false;
        if constexpr (C::PAIR) {
#pragma unroll
            for (int e = 0; e < NE; ++e) {
                const float2 a = v[0][e], b = v[1][e];
                *reinterpret_cast<float4*>(&dst[(size_t)(u[0] + e * Q) * W + w0]) =
                    CONJ ? make_float4(a.x, b.x, -a.y, -b.y) : make_float4(a.x, b.x, a.y, b.y);
            }
        } else {
#pragma unroll
            for (int s = 0; s < 2; ++s)
#pragma unroll
                for (int e = 0; e < 16; ++e)
                    if (!PAD || u[s] + e * Q < C::N / 2)
                        dst[u[s] + e * Q] = CONJ ? cconj(v[s][e]) : v[s][e];
        }
    }
}

template <int LOGN, int KIND, bool PAD, int MID, int IOM, bool X>
static cudaError_t launch_x(int n_tiles, cudaStream_t s, const PassParams& p) {
    // + two mbarriers + (packed column passes) the stage twiddles
    constexpr bool PACKED = !(KIND == ROW_FWD || KIND == ROW_INV) && Tile<LOGN>::PAIR && MID != MID_ASM_F64 && LOGN >= 8;
    constexpr size_t smem = ((X && KIND == ROW_FWD) ? Tile<LOGN>::SMEM_BYTES_X : Tile<LOGN>::SMEM_BYTES) + 64 +
                            (PACKED ? sizeof(float2) * PP<LOGN>::NTW_P : 0)
#ifdef CWO_FORCE_SMEM
                            + (PACKED ? CWO_FORCE_SMEM : 0)
#endif
        ;
    DeviceInfo* d = device_info();
    if (!d) return cudaErrorInvalidDevice;
    static FuncOnce once;
    if (!once.done(d->index)) {
        cudaError_t e = cudaFuncSetAttribute(pass_kernel<LOGN, KIND, PAD, MID, IOM, X>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        once.set(d->index);
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)n_tiles); cfg.blockDim = dim3((unsigned)Tile<LOGN>::T);
    cfg.dynamicSmemBytes = smem; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    // measured: early residency helps grids of a few waves (2048^2: 65.7 -> 63.2 us per propagation) and hurts
    // long ones (4096^2: 208.7 -> 221.9 us)
    at[0].val.programmaticStreamSerializationAllowed = n_tiles <= 1024 ? 1 : 0;
    cfg.attrs = at; cfg.numAttrs = 1;
    PassParams q = p;
    q.n_tiles = n_tiles;
    q.pf_dist = (!(KIND == ROW_FWD || KIND == ROW_INV) && p.n_planes <= 1) ? d->n_sm * Tile<LOGN>::MINB : 0;
    return cudaLaunchKernelEx(&cfg, pass_kernel<LOGN, KIND, PAD, MID, IOM, X>, q);
}

// pipe_kernel.cuh: persistent, prefetching form of the same pass for the HBM-sized tile shapes
constexpr bool pipe_supported(int logn) { return logn >= 10 && logn <= 12; }
template <int LOGN, int KIND, bool PAD, int MID, int IOM>
static cudaError_t launch_pipe(int n_tiles, cudaStream_t s, const PassParams& p);

// fold_kernel.cuh: pipelined inverse row pass of length 2n = 4096 / 8192 on one-row tiles (lane pair of the n-point transform)
constexpr bool fold_supported(int logn) { return logn == 12 || logn == 13; }
template <int LOGC, bool PAD>
static cudaError_t launch_fold(int n_rows, cudaStream_t s, const PassParams& p);

// cluster_kernel.cuh: forward row pass of 16384-point rows on 4-CTA clusters (32-byte workspace pieces)
constexpr int CLUSTER_LOGN = 14;
template <int LOGN, bool PAD>
static cudaError_t launch_cluster_row_fwd(int n_rows, cudaStream_t s, const PassParams& p);

// prefetch_kernel.cuh: fused column pass of the padded 8192/16384-point transforms, persistent with the next tile
// prefetched into a spare 64 KB buffer
constexpr size_t PREFETCH_BYTES = 65536;
template <int LOGN, int MID>
static cudaError_t launch_colpref(int n_tiles, cudaStream_t s, const PassParams& p);

// rowpair_kernel.cuh: forward row pass over 8192-point rows in packed arithmetic (one CTA per two-row tile)
constexpr int ROWPAIR_LOGN = 13;
template <int LOGN, bool PAD>
static cudaError_t launch_rowpair_fwd(int n_tiles, cudaStream_t s, const PassParams& p);

// colpad_kernel.cuh: fused column pass of the zero-expanded ASM on (even, odd)-bin lane pairs (zero half pruned)
constexpr bool colpad_supported(int logn) { return logn == 13; }   // (4096-point padded columns: 84.4 vs 78.8 us, not used)
template <int LOGN>
static cudaError_t launch_colpad_fused_asm(int n_tiles, cudaStream_t s, const PassParams& p);

// colfold_kernel.cuh: fused ASM column pass over 8192-point columns as (even, odd)-bin lane pairs (4 exchanges)
constexpr int COLFOLD_LOGN = 13;
template <int LOGN>
static cudaError_t launch_colfold_fused_asm(int n_tiles, cudaStream_t s, const PassParams& p);

template <int LOGN, int KIND, bool PAD, int MID, int IOM>
static cudaError_t launch_one(int n_tiles, cudaStream_t s, const PassParams& p) {
    if constexpr (LOGN == COLFOLD_LOGN && KIND == COL_FUSED && !PAD && MID == MID_ASM_SPLIT) {
        if (p.use_pipe && p.res_poly && !p.band && p.n_planes <= 1 && p.ly == Tile<LOGN>::N)
            return launch_colfold_fused_asm<LOGN>(n_tiles, s, p);
    }
    if constexpr (colpad_supported(LOGN) && KIND == COL_FUSED && PAD && MID == MID_ASM_SPLIT) {
        if (p.use_pipe && p.res_poly && !p.band && p.n_planes <= 1 && p.ly * 2 == Tile<LOGN>::N)
            return launch_colpad_fused_asm<LOGN>(n_tiles, s, p);
    }
    if constexpr (LOGN == ROWPAIR_LOGN && KIND == ROW_FWD && IOM == IN_COMPLEX) {
        if (p.use_pipe && p.logwc == 1 && p.rows % 2 == 0 && !p.use_cluster) return launch_rowpair_fwd<LOGN, PAD>(n_tiles, s, p);
    }
    if constexpr (KIND == COL_FUSED && PAD && MID != MID_ASM_F64 && LOGN >= 13) {
        if (p.use_pipe && (size_t)p.ly * Tile<LOGN>::W * 8 <= PREFETCH_BYTES) return launch_colpref<LOGN, MID>(n_tiles, s, p);
    }
    if constexpr (LOGN == CLUSTER_LOGN && KIND == ROW_FWD && IOM == IN_COMPLEX) {
        if (p.use_cluster) return launch_cluster_row_fwd<LOGN, PAD>(n_tiles, s, p);           // n_tiles = rows
    }
    constexpr bool ROWPASS = (KIND == ROW_FWD || KIND == ROW_INV);
    if constexpr (fold_supported(LOGN) && KIND == ROW_INV && IOM == OUT_COMPLEX) {
        if (p.use_fold) return launch_fold<LOGN - 1, PAD>(n_tiles, s, p);                     // n_tiles = rows
    }
#ifndef CWO_PIPE_FUSED
#define CWO_PIPE_FUSED 0
#endif
    if constexpr (pipe_supported(LOGN) && MID != MID_ASM_F64 && (CWO_PIPE_FUSED || KIND != COL_FUSED) &&
                  (!ROWPASS || (KIND == ROW_FWD && IOM == IN_COMPLEX) ||
                   (KIND == ROW_INV && (IOM == OUT_COMPLEX || IOM == OUT_INTENSITY || (IOM == OUT_PHASOR_AMP && !PAD))))) {
        if (p.use_pipe && (!ROWPASS || (p.use_tmap && p.rows % Tile<LOGN>::W == 0)))
            return launch_pipe<LOGN, KIND, PAD, MID, IOM>(n_tiles, s, p);
    }
    if constexpr ((KIND == ROW_FWD || KIND == ROW_INV) && Tile<LOGN>::W == 2) {
        if (p.logwc == 1) return launch_x<LOGN, KIND, PAD, MID, IOM, true>(n_tiles, s, p);
    }
    return launch_x<LOGN, KIND, PAD, MID, IOM, false>(n_tiles, s, p);
}

template <int LOGN, int KIND, bool PAD, int MID>
static cudaError_t launch_iom(int iom, int n_tiles, cudaStream_t s, const PassParams& p) {
    if constexpr (KIND == ROW_FWD) {
        return iom == IN_COMPLEX ? launch_one<LOGN, KIND, PAD, MID, IN_COMPLEX>(n_tiles, s, p)
                                 : launch_one<LOGN, KIND, PAD, MID, IN_AMP_PHASE>(n_tiles, s, p);
    } else if constexpr (KIND == ROW_INV) {
        return iom == OUT_COMPLEX      ? launch_one<LOGN, KIND, PAD, MID, OUT_COMPLEX>(n_tiles, s, p)
               : iom == OUT_PHASOR_AMP ? launch_one<LOGN, KIND, PAD, MID, OUT_PHASOR_AMP>(n_tiles, s, p)
               : iom == OUT_INTENSITY  ? launch_one<LOGN, KIND, PAD, MID, OUT_INTENSITY>(n_tiles, s, p)
                                       : launch_one<LOGN, KIND, PAD, MID, OUT_PHASE>(n_tiles, s, p);
    } else {
        return launch_one<LOGN, KIND, PAD, MID, 0>(n_tiles, s, p);
    }
}

template <int LOGN>
static cudaError_t launch_pass_impl(int kind, int pad, int mid, int n_tiles, cudaStream_t s, const PassParams& p) {
    const int key = kind * 100 + pad * 10 + mid;
    switch (key) {
        case ROW_FWD * 100 + 0: return launch_iom<LOGN, ROW_FWD, false, MID_NONE>(p.in_mode, n_tiles, s, p);
        case ROW_FWD * 100 + 10: return launch_iom<LOGN, ROW_FWD, true, MID_NONE>(p.in_mode, n_tiles, s, p);
        case ROW_INV * 100 + 0: return launch_iom<LOGN, ROW_INV, false, MID_NONE>(p.out_mode, n_tiles, s, p);
        case ROW_INV * 100 + 10: return launch_iom<LOGN, ROW_INV, true, MID_NONE>(p.out_mode, n_tiles, s, p);
        case COL_FWD * 100 + 0: return launch_iom<LOGN, COL_FWD, false, MID_NONE>(0, n_tiles, s, p);
        case COL_FUSED * 100 + 10 + MID_TABLES: return launch_iom<LOGN, COL_FUSED, true, MID_TABLES>(0, n_tiles, s, p);
        case COL_FUSED * 100 + MID_ASM_SPLIT: return launch_iom<LOGN, COL_FUSED, false, MID_ASM_SPLIT>(0, n_tiles, s, p);
        case COL_FUSED * 100 + MID_ASM_F64: return launch_iom<LOGN, COL_FUSED, false, MID_ASM_F64>(0, n_tiles, s, p);
        // zero-expanded ASM (CWO_OPT_ASM_PAD2X): the Fresnel pad/crop addressing with the ASM transfer function
        case COL_FUSED * 100 + 10 + MID_ASM_SPLIT: return launch_iom<LOGN, COL_FUSED, true, MID_ASM_SPLIT>(0, n_tiles, s, p);
        case COL_FUSED * 100 + 10 + MID_ASM_F64: return launch_iom<LOGN, COL_FUSED, true, MID_ASM_F64>(0, n_tiles, s, p);
        case COL_MIDINV * 100 + MID_ASM_SPLIT: return launch_iom<LOGN, COL_MIDINV, false, MID_ASM_SPLIT>(0, n_tiles, s, p);
        case COL_MIDINV * 100 + MID_ASM_F64: return launch_iom<LOGN, COL_MIDINV, false, MID_ASM_F64>(0, n_tiles, s, p);
    }
    return cudaErrorInvalidValue;
}

}  // namespace cwo
