// fft_packed.cuh -- the Stockham stages of fft_core.cuh on PACKED operands (sm_100a f32x2 arithmetic).
//
// A thread's two slots (the same 16-point unit in two adjacent lanes, fft_core.cuh) perform identical
// operations, so they are held as 64-bit register pairs, (slot 0, slot 1) of one real component, and
// every butterfly add/sub/constant rotation is ONE add/sub/mul/fma.f32x2 instruction for both slots.
// Packed instructions occupy the FMA pipe as long as the two scalar ones they replace, but take half the
// issue slots -- and issue slots, not HBM, are what bounds the fused column pass (profiles/).
// Stage twiddles are shared by the two slots, so their powers and products stay scalar (a packed power
// would compute the same number twice); scalar instructions address the halves of a pair directly.
// Arithmetic per sample is that of fft_core.cuh: same operations, same order, same rounding.
#pragma once
#include "fft_core.cuh"

namespace cwo {

typedef unsigned long long pk;   // two floats: low half = slot 0, high half = slot 1

__device__ __forceinline__ pk pk_make(float lo, float hi) {
    pk r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void pk_split(pk v, float& lo, float& hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ pk add2(pk a, pk b) { pk r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ pk sub2(pk a, pk b) { pk r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ pk mul2(pk a, pk b) { pk r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ pk fma2(pk a, pk b, pk c) {
    pk r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ pk pk_bcast(float c) { return pk_make(c, c); }   // folds into an .F32 (broadcast) operand
// sign flip of both halves; ptxas folds it into the operand modifiers of the FFMA2 / FADD2 / FMUL2 that consumes it
__device__ __forceinline__ pk pk_neg(pk a) {
    pk r;
    asm("{\n\t.reg .f32 lo, hi;\n\tmov.b64 {lo, hi}, %1;\n\tneg.f32 lo, lo;\n\tneg.f32 hi, hi;\n\tmov.b64 %0, {lo, hi};\n\t}"
        : "=l"(r) : "l"(a));
    return r;
}

// 16 complex points x 2 slots
struct PV { pk r[16], i[16]; };

// ---- in-register DFTs on elements b + k*S (same conventions and output positions as fft_core.cuh) ----
template <int S> __device__ __forceinline__ void dft2p(PV& v, int b) {
    const pk ar = v.r[b], ai = v.i[b], br = v.r[b + S], bi = v.i[b + S];
    v.r[b] = add2(ar, br); v.i[b] = add2(ai, bi);
    v.r[b + S] = sub2(ar, br); v.i[b + S] = sub2(ai, bi);
}

template <int S> __device__ __forceinline__ void dft4p(PV& v, int b) {   // natural order
    const pk ar = add2(v.r[b], v.r[b + 2 * S]), ai = add2(v.i[b], v.i[b + 2 * S]);
    const pk cr = sub2(v.r[b], v.r[b + 2 * S]), ci = sub2(v.i[b], v.i[b + 2 * S]);
    const pk er = add2(v.r[b + S], v.r[b + 3 * S]), ei = add2(v.i[b + S], v.i[b + 3 * S]);
    const pk tr = sub2(v.r[b + S], v.r[b + 3 * S]), ti = sub2(v.i[b + S], v.i[b + 3 * S]);
    // d = t * (-i) = (t.i, -t.r):  c + d = (c.r + t.i, c.i - t.r),  c - d = (c.r - t.i, c.i + t.r)
    v.r[b] = add2(ar, er); v.i[b] = add2(ai, ei);
    v.r[b + 2 * S] = sub2(ar, er); v.i[b + 2 * S] = sub2(ai, ei);
    v.r[b + S] = add2(cr, ti); v.i[b + S] = sub2(ci, tr);
    v.r[b + 3 * S] = sub2(cr, ti); v.i[b + 3 * S] = add2(ci, tr);
}

// x * (c8, -c8) = c8 (x.r + x.i, x.i - x.r);  x * (-c8, -c8) = c8 (x.i - x.r), -c8 (x.r + x.i)
__device__ __forceinline__ void rot_m2(PV& v, int k, pk c8) {
    const pk r = v.r[k], i = v.i[k];
    v.r[k] = mul2(add2(r, i), c8); v.i[k] = mul2(sub2(i, r), c8);
}
__device__ __forceinline__ void rot_m6(PV& v, int k, pk c8, pk nc8) {
    const pk r = v.r[k], i = v.i[k];
    v.r[k] = mul2(sub2(i, r), c8); v.i[k] = mul2(add2(r, i), nc8);
}
// x * (-i) = (x.i, -x.r)
__device__ __forceinline__ void rot_m4(PV& v, int k) {
    const pk r = v.r[k];
    v.r[k] = v.i[k]; v.i[k] = sub2(0ull, r);
}
// x * (a, b) with the constant given as packed a, b and -b:  (x.r a - x.i b, x.i a + x.r b)
__device__ __forceinline__ void rot_c(PV& v, int k, pk a, pk b, pk nb) {
    const pk r = v.r[k], i = v.i[k];
    v.r[k] = fma2(r, a, mul2(i, nb)); v.i[k] = fma2(i, a, mul2(r, b));
}

// 8 = 4 x 2 (fft_core.cuh dft8)
template <int S> __device__ __forceinline__ void dft8p(PV& v, int b) {
    const pk c8 = pk_bcast(CWO_C8), nc8 = pk_bcast(-CWO_C8);
    dft4p<2 * S>(v, b);
    dft4p<2 * S>(v, b + S);
    rot_m2(v, b + 3 * S, c8);
    rot_m4(v, b + 5 * S);
    rot_m6(v, b + 7 * S, c8, nc8);
#pragma unroll
    for (int q2 = 0; q2 < 4; ++q2) dft2p<S>(v, b + 2 * q2 * S);
}

// 16 = 4 x 4 (fft_core.cuh dft16): w16^m = (cos(pi m/8), -sin(pi m/8))
__device__ __forceinline__ void dft16p(PV& v) {
    const pk c8 = pk_bcast(CWO_C8), nc8 = pk_bcast(-CWO_C8);
    const pk c16 = pk_bcast(CWO_C16), nc16 = pk_bcast(-CWO_C16), s16 = pk_bcast(CWO_S16), ns16 = pk_bcast(-CWO_S16);
#pragma unroll
    for (int r1 = 0; r1 < 4; ++r1) dft4p<4>(v, r1);
    rot_c(v, 5, c16, ns16, s16);      // m = 1: (c16, -s16)
    rot_m2(v, 6, c8);                 // m = 2
    rot_c(v, 7, s16, nc16, c16);      // m = 3: (s16, -c16)
    rot_m2(v, 9, c8);                 // m = 2
    rot_m4(v, 10);                    // m = 4
    rot_m6(v, 11, c8, nc8);           // m = 6
    rot_c(v, 13, s16, nc16, c16);     // m = 3
    rot_m6(v, 14, c8, nc8);           // m = 6
    rot_c(v, 15, nc16, s16, ns16);    // m = 9: (-c16, s16)
#pragma unroll
    for (int q2 = 0; q2 < 4; ++q2) dft4p<1>(v, 4 * q2);
}

template <int R> __device__ __forceinline__ void dftRp(PV& v, int b) {
    if constexpr (R == 16) dft16p(v);
    else if constexpr (R == 8) dft8p<2>(v, b);
    else if constexpr (R == 4) dft4p<4>(v, b);
    else dft2p<8>(v, b);
}

// element k of both slots times the scalar twiddles w0 (slot 0) and w1 (slot 1)
__device__ __forceinline__ void mul_tw(PV& v, int k, float2 w0, float2 w1) {
    float r0, r1, i0, i1;
    pk_split(v.r[k], r0, r1); pk_split(v.i[k], i0, i1);
    const float2 a = cmul(make_float2(r0, i0), w0), b = cmul(make_float2(r1, i1), w1);
    v.r[k] = pk_make(a.x, b.x); v.i[k] = pk_make(a.y, b.y);
}
// element k of both slots times ONE twiddle w: packed multiplies with the scalar broadcast to both halves
// (SASS: FMUL2/FFMA2 with an .F32 operand -- no move, no second multiply); values as cmul()
__device__ __forceinline__ void mul_tw1(PV& v, int k, float2 w) {
    const pk r = v.r[k], i = v.i[k];
    v.r[k] = fma2(r, pk_bcast(w.x), mul2(i, pk_bcast(-w.y)));
    v.i[k] = fma2(r, pk_bcast(w.y), mul2(i, pk_bcast(w.x)));
}

template <int R> __device__ __forceinline__ void unpermute_p(PV& v) {
    constexpr int S = 16 / R;
    pk tr[16], ti[16];
#pragma unroll
    for (int e = 0; e < 16; ++e) { tr[e] = v.r[e]; ti[e] = v.i[e]; }
#pragma unroll
    for (int i = 0; i < S; ++i)
#pragma unroll
        for (int q = 0; q < R; ++q) { v.r[i + q * S] = tr[i + perm<R>(q) * S]; v.i[i + q * S] = ti[i + perm<R>(q) * S]; }
}

// w32^e = exp(-i 2 pi e/32), e = 0..15: the twiddle of point x = us + e*Q (Q = n/16) is w^us * w32^e.
// e is a compile-time constant after unrolling, so the table folds into immediates.
__device__ __forceinline__ float2 w32_pow(int e) {
    constexpr float c[16] = {1.0f, 0.98078528040323044913f, 0.92387953251128675613f, 0.83146961230254523708f,
                             0.70710678118654752440f, 0.55557023301960222474f, 0.38268343236508977173f,
                             0.19509032201612826785f, 0.0f, -0.19509032201612826785f, -0.38268343236508977173f,
                             -0.55557023301960222474f, -0.70710678118654752440f, -0.83146961230254523708f,
                             -0.92387953251128675613f, -0.98078528040323044913f};
    constexpr float sn[16] = {0.0f, 0.19509032201612826785f, 0.38268343236508977173f, 0.55557023301960222474f,
                              0.70710678118654752440f, 0.83146961230254523708f, 0.92387953251128675613f,
                              0.98078528040323044913f, 1.0f, 0.98078528040323044913f, 0.92387953251128675613f,
                              0.83146961230254523708f, 0.70710678118654752440f, 0.55557023301960222474f,
                              0.38268343236508977173f, 0.19509032201612826785f};
    return make_float2(c[e], -sn[e]);
}

// w16^i = exp(-i 2 pi i/16), i = 0..7 (compile-time index after unrolling: folds into immediates)
__device__ __forceinline__ float2 w16_pow(int i) {
    constexpr float c[8] = {1.0f, CWO_C16, CWO_C8, CWO_S16, 0.0f, -CWO_S16, -CWO_C8, -CWO_C16};
    constexpr float sn[8] = {0.0f, CWO_S16, CWO_C8, CWO_C16, 1.0f, CWO_C16, CWO_C8, CWO_S16};
    return make_float2(c[i], -sn[i]);
}

// Twiddle (if lns > 0) and butterflies of one radix-2^LR stage; both slots are unit `us` (shared twiddles).
// tw: shared-memory copy of the twiddle table (pipe_kernel.cuh).
// war: an exchange follows directly; its write-after-read synchronisation is taken here, between the twiddles
// and the butterflies, so that the exchange's stores can be scheduled among the butterflies.
template <int LOGN, int LR, class SY>
__device__ __forceinline__ void butterflies_p(PV& v, int us, int lns, const float2* tw, const SY& sync, bool war) {
    using C = Tile<LOGN>;
    constexpr int R = 1 << LR, S = 16 / R;
#pragma unroll
    for (int i = 0; i < S; ++i) {
        if (lns > 0) {
            float2 w[16];
            if (LR == 1 && lns == LOGN - 1) {
                // last stage of n = 2 * 16^m: the twiddle of unit us + i Q is w^us w16^i (Q = n/16), so that only the
                // first Q table entries are ever read (the shared-memory copy of the table holds just those)
                w[1] = i == 0 ? tw[us] : cmul(tw[us], w16_pow(i));
            } else {
                const int k0 = (us + i * C::Q) & ((1 << lns) - 1);
                powers<R>(tw[k0 << (LOGN - lns - LR)], w);
            }
#pragma unroll
            for (int r = 1; r < R; ++r) mul_tw1(v, i + r * S, w[r]);
        }
        if (SY::EARLY_WAR && war && i == 0) sync.war();
        dftRp<R>(v, i);
    }
}

// Exchange through shared memory, Stockham order (fft_core.cuh exchange()); one 16-byte element
// (r.slot0, r.slot1, i.slot0, i.slot1) per point and lane pair, one pad row every 16 points.
// The padded index of point j0 + q*2^lns is affine in q when lns == 0 (j0 is a multiple of 2^LR = 16) or
// lns >= 4, and that of point us + e*Q is affine in e (Q is a multiple of 16): one address computation per
// unit, immediate offsets per access.
// LOGW: log2 of the lanes of the tile (default: the tile shape of the length; the 8192-point forward row pass runs
// 4096-point lanes on a four-lane tile)
template <int LOGN, int LR, class SY, int LOGW = tile_logw(LOGN)>
__device__ __forceinline__ void exchange_store_p(const PV& v, int us, int w0, int lns, float2* sm, const SY& sync) {
    using C = Tile<LOGN>;
    constexpr int R = 1 << LR, S = 16 / R, H = (1 << LOGW) / 2;
    ulonglong2* rg = reinterpret_cast<ulonglong2*>(sm);
    const int wh = w0 >> 1;
    if (!SY::EARLY_WAR) sync.war();                       // else taken by butterflies_p (war = true)
#pragma unroll
    for (int i = 0; i < S; ++i) {
        const int j = us + i * C::Q;
        const int j0 = ((j >> lns) << (lns + LR)) + (j & ((1 << lns) - 1));
        ulonglong2* b = rg + (j0 + (j0 >> 4)) * H + wh;
        if (LR == 4 && lns == 0) {
#pragma unroll
            for (int q = 0; q < R; ++q) b[q * H] = make_ulonglong2(v.r[i + perm<R>(q) * S], v.i[i + perm<R>(q) * S]);
        } else if (lns >= 4) {
            const int st = (17 << (lns - 4)) * H;             // (2^lns + 2^lns / 16) * H
#pragma unroll
            for (int q = 0; q < R; ++q) b[q * st] = make_ulonglong2(v.r[i + perm<R>(q) * S], v.i[i + perm<R>(q) * S]);
        } else {
#pragma unroll
            for (int q = 0; q < R; ++q) {
                const int p = j0 + (q << lns);
                rg[(p + (p >> 4)) * H + wh] = make_ulonglong2(v.r[i + perm<R>(q) * S], v.i[i + perm<R>(q) * S]);
            }
        }
    }
}
template <int LOGN, class SY, int LOGW = tile_logw(LOGN)>
__device__ __forceinline__ void exchange_load_p(PV& v, int us, int w0, const float2* sm, const SY& sync) {
    using C = Tile<LOGN>;
    constexpr int H = (1 << LOGW) / 2;
    const ulonglong2* rg = reinterpret_cast<const ulonglong2*>(sm);
    const int wh = w0 >> 1;
    static_assert(C::Q % 16 == 0, "Q multiple of 16");
    const ulonglong2* b = rg + (us + (us >> 4)) * H + wh;
#pragma unroll
    for (int e = 0; e < 16; ++e) {
        const ulonglong2 t = b[e * (C::Q + C::Q / 16) * H];
        v.r[e] = t.x; v.i[e] = t.y;
    }
    sync.consumed();
}
template <int LOGN, int LR, class SY, int LOGW = tile_logw(LOGN)>
__device__ __forceinline__ void exchange_p(PV& v, int us, int w0, int lns, float2* sm, const SY& sync) {
    exchange_store_p<LOGN, LR, SY, LOGW>(v, us, w0, lns, sm, sync);
    sync.raw();
    exchange_load_p<LOGN, SY, LOGW>(v, us, w0, sm, sync);
}

// radix-16 stage with the twiddle powers w[1..15] supplied (computed during the previous exchange)
template <int LOGN, class SY>
__device__ __forceinline__ void butterflies16_p(PV& v, int lns, const float2 (&w)[16], const SY& sync, bool war) {
    if (lns > 0) {
#pragma unroll
        for (int r = 1; r < 16; ++r) mul_tw1(v, r, w[r]);
    }
    if (SY::EARLY_WAR && war) sync.war();
    dft16p(v);
}
template <int LOGN>
__device__ __forceinline__ void stage_powers(int us, int lns, const float2* tw, float2 (&w)[16]) {
    if (lns > 0) powers<16>(tw[(us & ((1 << lns) - 1)) << (LOGN - lns - 4)], w);
}

// transform_p for split-phase synchronisation (SyncSplit): the twiddle powers of stage s + 1 are formed inside
// the exchange after stage s.  Otherwise as transform_p below.
// Forward and/or inverse transform of the tile held in registers (fft_core.cuh transform()).  `mid`
// (mid.packed(v), which must also conjugate) runs between the two, or first when MID_FIRST.  The last
// forward stage, mid and the first inverse stage (no twiddles) form one compute phase without an exchange.
template <int LOGN, bool HAS_FWD, bool HAS_INV, bool MID_FIRST, class Mid, class SY, int LOGW = tile_logw(LOGN)>
__device__ __forceinline__ void transform_ahead_p(PV& v, int us, int w0, float2* sm, const float2* tw, const Mid& mid,
                                            const SY& sync) {
    using C = Tile<LOGN>;
    constexpr int L0 = C::L0, M = C::M;
    static_assert(!(HAS_FWD && HAS_INV) || M >= 2, "merged middle phase needs an exchange after it");
    if constexpr (HAS_FWD && L0 > 0) {
        butterflies_p<LOGN, L0>(v, us, 0, tw, sync, true);
        exchange_p<LOGN, L0, SY, LOGW>(v, us, w0, 0, sm, sync);
    }
    constexpr int NST = (HAS_FWD ? M : 0) + (HAS_INV ? M : 0);
    // Ns = 2^lns of radix-16 stage s of the list [forward 0..M-1 | inverse M..2M-1]
    auto lns_of = [](int s) { return (HAS_FWD && s < M) ? L0 + 4 * s : 4 * (HAS_FWD ? s - M : s); };
    float2 w[16];
    stage_powers<LOGN>(us, lns_of(0), tw, w);
#pragma unroll 1
    for (int s = 0; s < NST; ++s) {
        const bool inv_half = HAS_FWD ? (s >= M) : true;
        const int sl = (HAS_FWD && inv_half) ? s - M : s;
        int lns = lns_of(s);
        const bool fwd_end = !inv_half && sl == M - 1;       // no exchange directly after these butterflies
        const bool inv_end = inv_half && sl == M - 1 && L0 == 0;
        if (MID_FIRST && s == 0) mid.packed(v);
        butterflies16_p<LOGN>(v, lns, w, sync, !fwd_end && !inv_end);
        if (fwd_end) {                                       // end of the forward transform
            unpermute_p<16>(v);
            if constexpr (!HAS_INV) break;
            mid.packed(v);
            butterflies16_p<LOGN>(v, 0, w, sync, true);      // first inverse stage (no twiddles), same phase
            ++s; lns = 0;
        } else if (inv_end) {                                // end of the inverse transform
            unpermute_p<16>(v);
            break;
        }
        // exchange; the next stage's twiddle powers are formed between publishing the stores and waiting for
        // everybody else's (they need neither, and v is dead in between)
        exchange_store_p<LOGN, 4, SY, LOGW>(v, us, w0, lns, sm, sync);
        sync.raw_arrive();
        if (s + 1 < NST) stage_powers<LOGN>(us, lns_of(s + 1), tw, w);
        sync.raw_wait();
        exchange_load_p<LOGN, SY, LOGW>(v, us, w0, sm, sync);
    }
    if constexpr (HAS_INV && L0 > 0) {
        butterflies_p<LOGN, L0>(v, us, 4 * M, tw, sync, false);
        unpermute_p<(1 << L0)>(v);
    }
}

// Forward and/or inverse transform of the tile held in registers (fft_core.cuh transform()).  `mid`
// (mid.packed(v), which must also conjugate) runs between the two, or first when MID_FIRST.  The last
// forward stage, mid and the first inverse stage (no twiddles) form one compute phase without an exchange.
template <int LOGN, bool HAS_FWD, bool HAS_INV, bool MID_FIRST, class Mid, class SY, int LOGW = tile_logw(LOGN)>
__device__ __forceinline__ void transform_p(PV& v, int us, int w0, float2* sm, const float2* tw, const Mid& mid,
                                            const SY& sync) {
    using C = Tile<LOGN>;
    constexpr int L0 = C::L0, M = C::M;
    static_assert(!(HAS_FWD && HAS_INV) || M >= 2, "merged middle phase needs an exchange after it");
    if constexpr (SY::EARLY_WAR) {
        transform_ahead_p<LOGN, HAS_FWD, HAS_INV, MID_FIRST, Mid, SY, LOGW>(v, us, w0, sm, tw, mid, sync);
        return;
    }
    if constexpr (HAS_FWD && L0 > 0) {
        butterflies_p<LOGN, L0>(v, us, 0, tw, sync, true);
        exchange_p<LOGN, L0, SY, LOGW>(v, us, w0, 0, sm, sync);
    }
    constexpr int NST = (HAS_FWD ? M : 0) + (HAS_INV ? M : 0);
#pragma unroll 1
    for (int s = 0; s < NST; ++s) {
        const bool inv_half = HAS_FWD ? (s >= M) : true;
        const int sl = (HAS_FWD && inv_half) ? s - M : s;
        int lns = inv_half ? 4 * sl : L0 + 4 * sl;
        const bool fwd_end = !inv_half && sl == M - 1;       // no exchange directly after these butterflies
        const bool inv_end = inv_half && sl == M - 1 && L0 == 0;
        if (MID_FIRST && s == 0) mid.packed(v);
        butterflies_p<LOGN, 4>(v, us, lns, tw, sync, !fwd_end && !inv_end);
        if (fwd_end) {                                       // end of the forward transform
            unpermute_p<16>(v);
            if constexpr (!HAS_INV) break;
            mid.packed(v);
            butterflies_p<LOGN, 4>(v, us, 0, tw, sync, true);   // first inverse stage, same phase
            ++s; lns = 0;
        } else if (inv_end) {                                // end of the inverse transform
            unpermute_p<16>(v);
            break;
        }
        exchange_p<LOGN, 4, SY, LOGW>(v, us, w0, lns, sm, sync);
    }
    if constexpr (HAS_INV && L0 > 0) {
        butterflies_p<LOGN, L0>(v, us, 4 * M, tw, sync, false);
        unpermute_p<(1 << L0)>(v);
    }
}

}  // namespace cwo
