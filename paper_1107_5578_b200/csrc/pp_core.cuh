// pp_core.cuh -- "ping-pong" scheduling of the Stockham stages of fft_core.cuh.
//
// A thread owns two slots (the same unit in two adjacent lanes).  Instead of exchanging both slots
// through shared memory at once (all warps store, barrier, all warps load: the FMA pipes idle while the
// shared-memory pipe works and vice versa), the two slots run half a stage apart:
//
//     cB(k); bar; ldsA; stsB(k); cA(k+1); bar; ldsB; stsA(k+1); cB(k+1); ...
//
// so every store is followed by a whole butterfly block of the other slot before the barrier that
// publishes it, and shared-memory traffic is spread evenly between the FMA work of every warp.
// Slot A (even lanes) and slot B (odd lanes) live in separate regions [point][W/2 lanes], one pad
// element row every 16 points.  `tw` is the CTA's shared-memory copy of the first PP::NTW twiddles (every
// index used by a stage is below N/16, or below 16^M for the small inverse radix): plain loads, no __ldg.  Arithmetic and operation order per sample are those of transform().
#pragma once
#include "fft_core.cuh"

namespace cwo {

// element index of (point p, lane pair wh) inside a slot region
template <int LOGN> __device__ __forceinline__ int ridx(int p, int wh) {
    return (p + (p >> 4)) * (Tile<LOGN>::W / 2) + wh;
}
template <int LOGN> struct PP {
    static constexpr int REGION = (Tile<LOGN>::N + Tile<LOGN>::N / 16) * (Tile<LOGN>::W / 2);   // elements
    // twiddles a CTA keeps in shared memory: indices < N/16 for radix-16 stages, < 16^M for the small inverse radix
    static constexpr int NTW = Tile<LOGN>::L0 == 0 ? Tile<LOGN>::Q : (1 << (4 * Tile<LOGN>::M));
    // the packed transforms (fft_packed.cuh) form the last radix-2 twiddles from the first Q entries
    static constexpr int NTW_P = Tile<LOGN>::L0 <= 1 ? Tile<LOGN>::Q : (1 << (4 * Tile<LOGN>::M));
};

// outputs of a radix-2^LR stage with Ns = 2^lns, one slot, Stockham order.  The padded index of
// point j0 + q*2^lns is affine in q when lns == 0 (j0 is a multiple of 2^LR) or lns >= 4, so those
// cases cost one address computation per unit instead of one per store.
template <int LOGN, int LR>
__device__ __forceinline__ void sts_slot(const float2 (&v)[16], int us, int wh, int lns, float2* rg) {
    using C = Tile<LOGN>;
    constexpr int R = 1 << LR, S = 16 / R, H = C::W / 2;
#pragma unroll
    for (int i = 0; i < S; ++i) {
        const int j = us + i * C::Q;
        const int j0 = ((j >> lns) << (lns + LR)) + (j & ((1 << lns) - 1));
        if (lns == 0 && LR == 4) {
            float2* b = rg + ridx<LOGN>(j0, wh);            // j0 = 16 j: the 16 outputs share a pad row
#pragma unroll
            for (int q = 0; q < R; ++q) b[q * H] = v[i + perm<R>(q) * S];
        } else if (lns >= 4) {
            float2* b = rg + ridx<LOGN>(j0, wh);
            const int st = (17 << (lns - 4)) * H;            // (2^lns + 2^lns/16) * H
#pragma unroll
            for (int q = 0; q < R; ++q) b[q * st] = v[i + perm<R>(q) * S];
        } else {
#pragma unroll
            for (int q = 0; q < R; ++q) rg[ridx<LOGN>(j0 + (q << lns), wh)] = v[i + perm<R>(q) * S];
        }
    }
}

// inputs of the next stage: register e <-> point us + e*Q (Q is a multiple of 16: affine in e)
template <int LOGN>
__device__ __forceinline__ void lds_slot(float2 (&v)[16], int us, int wh, const float2* rg) {
    using C = Tile<LOGN>;
    static_assert(C::Q % 16 == 0, "Q multiple of 16");
    const float2* b = rg + ridx<LOGN>(us, wh);
#pragma unroll
    for (int e = 0; e < 16; ++e) v[e] = b[e * (C::Q + C::Q / 16) * (C::W / 2)];
}

// one small-radix stage (own twiddles) on one slot
template <int LOGN, int LR>
__device__ __forceinline__ void slot_small(float2 (&v)[16], int us, int lns, const float2* __restrict__ tw) {
    using C = Tile<LOGN>;
    constexpr int R = 1 << LR, S = 16 / R;
#pragma unroll
    for (int i = 0; i < S; ++i) {
        if (lns > 0) {
            float2 w[16];
            const int k0 = (us + i * C::Q) & ((1 << lns) - 1);
            powers<R>(tw[k0 << (LOGN - lns - LR)], w);
            apply_powers<R>(v, i, w);
        }
        dftR<R>(v, i);
    }
}

// Runs the radix-16 stages SA..SB-1 of the concatenated list [forward stages 0..M-1 | inverse stages
// M..2M-1] (forward stage s: Ns = 2^(L0+4s); inverse stage M+s: Ns = 2^(4s)), preceded by the small
// forward radix (FWD_SMALL) and followed by the small inverse radix (INV_SMALL) when L0 > 0.
// In:  both slots hold the inputs of the first block (register e <-> point us + e*Q); the regions are
//      free (callers put a barrier between their last use and this call).
// Out: outputs of the last block; after a radix-16 block they are still in dft16's permuted order.
template <int LOGN, bool FWD_SMALL, int SA, int SB, bool INV_SMALL, class SY>
__device__ __forceinline__ void pp_run(float2 (&v)[2][16], int us, int wh, float2* rgA, float2* rgB,
                                       const float2* __restrict__ tw, const SY& sync) {
    using C = Tile<LOGN>;
    constexpr int L0 = C::L0, M = C::M;
    bool pendB = false;                 // slot B's inputs are still in (or on their way to) its region
    if constexpr (FWD_SMALL && L0 > 0) {
        slot_small<LOGN, L0>(v[0], us, 0, tw);
        sts_slot<LOGN, L0>(v[0], us, wh, 0, rgA);
        slot_small<LOGN, L0>(v[1], us, 0, tw);
        sync();
        lds_slot<LOGN>(v[0], us, wh, rgA);
        sts_slot<LOGN, L0>(v[1], us, wh, 0, rgB);
        pendB = true;
    }
#pragma unroll 1
    for (int s = SA; s < SB;) {
        const bool inv_half = s >= M;
        const int lns = inv_half ? 4 * (s - M) : L0 + 4 * s;
        const int sn = s + 1;
        const bool has_next = (sn < SB) || (INV_SMALL && L0 > 0);
        const int lns_out = lns;
        const float2 w1 = tw[(us & ((1 << lns) - 1)) << (LOGN - lns - 4)];
#pragma unroll
        for (int sl = 0; sl < 2; ++sl) {
            if (lns > 0) {
                // powers rebuilt per slot: 15 fewer live complex registers across the exchange of the other slot
                float2 w[16];
                powers<16>(w1, w);
                apply_powers<16>(v[sl], 0, w);
            }
            dft16(v[sl]);
            if (sl == 0) {
                if (pendB) { sync(); lds_slot<LOGN>(v[1], us, wh, rgB); }
                if (has_next) sts_slot<LOGN, 4>(v[0], us, wh, lns_out, rgA);
            } else if (has_next) {
                sync();
                lds_slot<LOGN>(v[0], us, wh, rgA);
                sts_slot<LOGN, 4>(v[1], us, wh, lns_out, rgB);
                pendB = true;
            }
        }
        s = sn;
    }
    if constexpr (INV_SMALL && L0 > 0) {
        slot_small<LOGN, L0>(v[0], us, 4 * M, tw);
        sync();
        lds_slot<LOGN>(v[1], us, wh, rgB);
        slot_small<LOGN, L0>(v[1], us, 4 * M, tw);
        unpermute<(1 << L0)>(v[0]); unpermute<(1 << L0)>(v[1]);
    }
}

}  // namespace cwo
