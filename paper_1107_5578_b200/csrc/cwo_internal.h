// cwo_internal.h -- plan object, pass descriptors and launcher declarations shared by the
// translation units of libcwo.so.  Not part of the public ABI (see include/cwo.h).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>

namespace cwo {

// ---- how one streaming pass addresses global memory -----------------------------------------
// element offset of (tile, lane w, point p) =
//     tile*tile_stride + w*lane_stride + (p >> sh)*hi_stride + (p & mask)*lo_stride
// Row pass over a row-major field : lanes = rows, points = x : sh=0, hi=1, mask=0
// Row pass over the column-tiled ws: T[x/Wc][y][x%Wc]        : sh=log2 Wc, hi=Ly*Wc, mask=Wc-1, lo=1
// Column pass over the tiled ws   : lanes = columns in tile, points = y : sh=0, hi=Wc, mask=0
struct Addr {
    long long tile_stride;
    unsigned lane_stride, hi_stride, lo_stride;
    int sh, mask;
};

enum InMode { IN_COMPLEX = 0, IN_AMP_PHASE = 1 };
enum OutMode { OUT_COMPLEX = 0, OUT_PHASOR_AMP = 1, OUT_PHASE = 2 };
enum MidMode { MID_NONE = 0, MID_ASM_F64 = 1, MID_TABLES = 2, MID_ASM_SPLIT = 3 };
enum Kind { KIND_FWD = 0, KIND_INV = 1, KIND_FUSED = 2, KIND_MIDINV = 3, KIND_COUNT = 4 };

struct PassParams {
    const float2* in;
    float2* out;              // OUT_PHASE: float*
    const float* in_amp;      // IN_AMP_PHASE: amplitude [rows][aux_pitch]
    const float* in_phase;    //               phase
    const float* out_amp;     // OUT_PHASOR_AMP: amplitude of the next plane
    Addr ain, aout;
    int in_mode, out_mode, mid_mode;
    int aux_pitch;            // row pitch (elements) of the real arrays
    int p_in_valid;           // points >= this load as 0 (zero padding folded into addressing, S3)
    int p_out_valid;          // points >= this are not stored (crop folded into addressing, S8)
    int lanes_total;          // lanes beyond this are masked (tile overhang on tiny fields)
    const float2* tw;         // forward twiddles exp(-i 2 pi m/n), m < n
    float out_scale;          // applied by the store
    // MID (transfer function / impulse-response spectrum, S2/S5/S7)
    double z, inv_lam2, df_lane, df_point;   // ASM: H from fp64 phase; lane = x bin, point = y bin
    int n_lane_bins;                          // Mx (for the signed-bin map of the lane index)
    float mid_scale;
    const float2* tab_lane;   // MID_TABLES: Cx[k];  MID_ASM_SPLIT: Ex[k]*c0
    const float2* tab_point;  // MID_TABLES: Cy[l];  MID_ASM_SPLIT: Ey[l]
    float res_a, res_b, res_c;  // MID_ASM_SPLIT residual constants
};

// per-length tile configuration (kept in one place: host sizing and kernels must agree)
constexpr int tile_logw(int logn) {
    return logn <= 9 ? 4 : logn == 10 ? 3 : logn == 11 ? 2 : logn == 12 ? 1 : logn == 13 ? 1 : 0;
}
constexpr int tile_threads(int logn) {
    // units = (n/16)*W ; threads = units / UPT
    return logn <= 5 ? 32 : logn == 6 ? 64 : logn == 7 ? 128 : logn <= 12 ? 256 : 512;
}
constexpr int tile_upt(int logn) { return (((1 << logn) / 16) << tile_logw(logn)) / tile_threads(logn); }
constexpr int tile_minblocks(int logn) { return logn <= 12 ? 2 : 1; }

constexpr int MIN_LOGN = 5, MAX_LOGN = 14;

// one launcher per transform length, defined in pass_inst.cu compiled with -DCWO_LOGN=<k>
typedef cudaError_t (*pass_launcher_t)(int kind, int n_tiles, cudaStream_t s, const PassParams& p);
#define CWO_DECL_LAUNCH(k) cudaError_t launch_pass_##k(int kind, int n_tiles, cudaStream_t s, const PassParams& p);
CWO_DECL_LAUNCH(5) CWO_DECL_LAUNCH(6) CWO_DECL_LAUNCH(7) CWO_DECL_LAUNCH(8) CWO_DECL_LAUNCH(9)
CWO_DECL_LAUNCH(10) CWO_DECL_LAUNCH(11) CWO_DECL_LAUNCH(12) CWO_DECL_LAUNCH(13) CWO_DECL_LAUNCH(14)
#undef CWO_DECL_LAUNCH

// tables.cu
cudaError_t build_twiddles(float2* tw, int n, cudaStream_t s);                 // exp(-i 2 pi m/n), fp64 -> fp32
cudaError_t build_twiddles_f64(double2* tw, int n, cudaStream_t s);            // same, kept in fp64, m < n/2
// Fresnel: spectrum of the sampled 1-D chirp, C[k] = coef * sum_{d=-N}^{N-1} exp(i pi (d pitch)^2/(lambda z)) exp(-i 2 pi dk/M)
// for up to two axes in one launch (axis 1 skipped when out1 == nullptr).  scratch: 2*M double2 per axis.
struct ChirpAxis { float2* out; double2* scratch; const double2* tw64; int logm; double a_cycles; double2 coef; };
cudaError_t build_chirp_spectrum(const ChirpAxis& ax0, const ChirpAxis* ax1, cudaStream_t s);

}  // namespace cwo
