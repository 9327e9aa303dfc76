// cwo_internal.h -- pass descriptors and launcher declarations shared by the translation units
// of libcwo.so.  Not part of the public ABI (see include/cwo.h).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stddef.h>
#include <atomic>

namespace cwo {

enum InMode { IN_COMPLEX = 0, IN_AMP_PHASE = 1 };
enum OutMode { OUT_COMPLEX = 0, OUT_PHASOR_AMP = 1, OUT_PHASE = 2, OUT_INTENSITY = 3 };
// the real fields of section 5 an OUT_INTENSITY store can write; REAL_PHASE only in the transposing store
enum RealMode { REAL_ABS2 = 0, REAL_ABS = 1, REAL_RE = 2, REAL_IM = 3, REAL_PHASE = 4 };
#ifdef __CUDACC__
// real field of the sample (re - i mim) * sc, i.e. of the conjugate of (re, mim) as the inverse passes hold it
__device__ __forceinline__ float real_field(float re, float mim, float sc, int mode) {
    switch (mode) {
        case REAL_ABS: return sqrtf(re * re + mim * mim) * sc;
        case REAL_RE: return re * sc;
        case REAL_IM: return -mim * sc;
        case REAL_PHASE: return (re == 0.0f && mim == 0.0f) ? 0.0f : atan2f(-mim, re);     // Eq.(25); phasor(0) = 1
        default: return (re * re + mim * mim) * (sc * sc);                                   // Eq.(20)
    }
}
#endif
enum MidMode { MID_NONE = 0, MID_TABLES = 1, MID_ASM_SPLIT = 2, MID_ASM_F64 = 3 };

struct PassParams {
    CUtensorMap tmap;         // pipelined row passes: the column-tiled workspace as a 2-D tensor (see encode_ws_tmap)
    int use_tmap;             // 1: tmap is valid, the row pass moves its workspace side with TMA tensor copies
    int use_cluster;          // 1: 16384-point forward row pass on 4-CTA clusters (cluster_kernel.cuh); tmap has 4-row boxes
    int use_fold;             // 1: 8192-point inverse row pass on one-row tiles (fold_kernel.cuh); tmap has one-row boxes
    const float2* in;
    float2* out;              // OUT_PHASE, OUT_INTENSITY: float*
    const float* in_amp;      // IN_AMP_PHASE: amplitude [rows][pitch]
    const float* in_phase;    //               phase
    const float* out_amp;     // OUT_PHASOR_AMP: amplitude of the next plane
    int in_mode, out_mode;
    int rows;                 // row passes: number of field rows (lanes beyond it are masked)
    int pitch;                // row passes: row pitch (elements) of the row-major field and real arrays
    int ly;                   // rows kept in the column-tiled workspace
    int logwc;                // row passes: log2 of the column-tile width of the workspace
    int n_tiles;              // total number of tiles
    int pf_dist;              // one-CTA-per-tile column passes: L2 prefetch distance in tiles (0: off)
    // batched planes (depth stack, pipelined kernels only): tile t belongs to plane t / tiles_per_plane
    int n_planes;             // 0 or 1: a single plane
    int tiles_per_plane;
    size_t in_plane_stride;   // complex elements between the planes of `in` (0: every plane reads the same data)
    size_t out_plane_stride;  // same for `out`
    int tab_plane_stride;     // MID_ASM_SPLIT: floats between the planes' [theta_x | theta_y] tables
    const float* plane_resc;  // MID_ASM_SPLIT: res_c (= z/lambda) of every plane
    int use_pipe;             // 1: use the pipelined form where it exists (CWO_OPT_PIPELINE)
    const float2* tw;         // forward twiddles exp(-i 2 pi m/n), m < n
    float out_scale;          // ROW_INV store
    int real_mode;            // OUT_INTENSITY store: which real field (RealMode; 0 = |u|^2)
    // Mid (transfer function / impulse-response spectrum, S2/S5/S7); lane = x bin, point = y bin
    double z, inv_lam2, df_lane, df_point;   // MID_ASM_F64
    int n_lane_bins;                          // Mx (signed-bin map of the lane index)
    const float2* tab_lane;   // MID_TABLES: Cx[k] (float2);  MID_ASM_SPLIT: theta_x[k] (float, cycles)
    const float2* tab_point;  // MID_TABLES: Cy[l];           MID_ASM_SPLIT: theta_y[l]
    float res_a, res_b, res_c;  // MID_ASM_SPLIT: lambda^2 dfx^2, lambda^2 dfy^2, z/lambda
    // shifted / band-limited angular spectrum method (Eq.(18)-(19), CWO_OPT_ASM_BAND_LIMIT): bins whose signed index is
    // outside [lo, hi] are zeroed; the phase ramp of Eq.(19) is in the theta tables (split) or formed from off_* (fp64)
    int band, band_lane_lo, band_lane_hi, band_point_lo, band_point_hi;
    double off_lane, off_point;
    int res_poly;               // MID_ASM_SPLIT: 1 = the degree-7 series of the residual is exact to 1e-7 cycles for every bin
};

constexpr int MIN_LOGN = 5, MAX_LOGN = 14;

// ---- per-device launch state ------------------------------------------------------------------------------
// A plan belongs to the device that was current when it was made; launch attributes (opt-in shared memory) and
// the SM count are per device, so the launchers cache them per device index, not per process.
struct DeviceInfo { int index, n_sm; };
constexpr int MAX_DEVICES = 64;
inline DeviceInfo* device_info() {                     // the current device; nullptr on error
    static DeviceInfo info[MAX_DEVICES];
    static std::atomic<int> known[MAX_DEVICES];
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= MAX_DEVICES) return nullptr;
    if (!known[dev].load(std::memory_order_acquire)) {
        int n = 0;
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) return nullptr;
        info[dev].index = dev; info[dev].n_sm = n;       // idempotent: a race writes the same values
        known[dev].store(1, std::memory_order_release);
    }
    return &info[dev];
}
// "cudaFuncSetAttribute has been called for this kernel on device d" (setting it twice is harmless)
struct FuncOnce {
    std::atomic<unsigned long long> mask{0};
    bool done(int dev) const { return (mask.load(std::memory_order_acquire) >> dev) & 1ull; }
    void set(int dev) { mask.fetch_or(1ull << dev, std::memory_order_release); }
};

// ---- separable Fresnel convolution (lineconv_kernel.cuh) ---------------------------------------------------
struct ConvParams {
    const float2* in;          // [n_lines][N] complex; gather: sample n of line l at in[n * in_stride + l] (the lines are the
                               // COLUMNS of a row-major [N][in_stride] field: no transpose between the two axes' passes)
    int gather, in_stride;
    const float* in_amp;       // variant 1: amplitude and phase, [n_lines][N]
    const float* in_phase;
    void* out;                 // [n_lines][N] complex, or float phase (variant 3); may alias `in`
    const float* mid_amp;      // variant 2: amplitude imposed between the two convolutions, [n_lines][N]
    const ulonglong2* tab[2];  // spectrum of the sampled chirp for convolution 0 / 1, planar pairs, N entries
    const float2* pre;         // variant 4: factor on every input sample, N entries (Eq.(12))
    const float2* post;        // variant 4: factor on every output sample, N entries (Eq.(11))
    const float2* tw;          // N-point forward twiddles
    const float2* tw2;         // 2N-point forward twiddles
    int n_lines;
    int n_tiles;
    int pf_dist;               // one CTA per tile: tiles between a CTA and the one that replaces it on its SM
    int* counter;              // persistent form: {next tile, CTAs done}, zero between launches (self-resetting)
};
// variant: 0 complex -> conv -> complex; 1 amp, phase -> conv -> complex; 2 complex -> conv, GS constraint, conv -> complex;
//          3 complex -> conv -> phase; 4 complex -> x pre -> conv -> x post -> complex (shifted Fresnel)
typedef cudaError_t (*conv_launcher_t)(int variant, cudaStream_t s, const ConvParams& p);

// one launcher per transform length, defined in pass_inst.cu compiled with -DCWO_LOGN=<k>
typedef cudaError_t (*pass_launcher_t)(int kind, int pad, int mid, int n_tiles, cudaStream_t s, const PassParams& p);
#define CWO_DECL_LAUNCH(k) \
    cudaError_t launch_pass_##k(int kind, int pad, int mid, int n_tiles, cudaStream_t s, const PassParams& p);
CWO_DECL_LAUNCH(5) CWO_DECL_LAUNCH(6) CWO_DECL_LAUNCH(7) CWO_DECL_LAUNCH(8) CWO_DECL_LAUNCH(9)
CWO_DECL_LAUNCH(10) CWO_DECL_LAUNCH(11) CWO_DECL_LAUNCH(12) CWO_DECL_LAUNCH(13) CWO_DECL_LAUNCH(14)
#undef CWO_DECL_LAUNCH
// lane-pair lengths 256..8192: separable Fresnel line convolution
#define CWO_DECL_LAUNCH(k) cudaError_t launch_conv_##k(int variant, cudaStream_t s, const ConvParams& p);
CWO_DECL_LAUNCH(8) CWO_DECL_LAUNCH(9) CWO_DECL_LAUNCH(10) CWO_DECL_LAUNCH(11) CWO_DECL_LAUNCH(12) CWO_DECL_LAUNCH(13)
#undef CWO_DECL_LAUNCH
constexpr int MIN_PAIR_LOGN = 8, MAX_PAIR_LOGN = 13;

// ---- line transforms of the Fourier-form Fresnel diffraction (linefft_kernel.cuh) ---------------------------
// out[line][k] = post[k] * DFT_N(pre[j] * in[line][j])[k]  (inverse != 0: the unnormalised inverse kernel); may run in place
struct LineFftParams {
    const float2* in; float2* out;
    const float2* pre; const float2* post;     // N entries each
    const float2* tw;                          // N-point forward twiddles
    int n_lines, inverse;
    int pf_dist;                               // tiles between a CTA and the one that replaces it on its SM
};
#define CWO_DECL_LAUNCH(k) cudaError_t launch_linefft_##k(cudaStream_t s, const LineFftParams& p);
CWO_DECL_LAUNCH(8) CWO_DECL_LAUNCH(9) CWO_DECL_LAUNCH(10) CWO_DECL_LAUNCH(11) CWO_DECL_LAUNCH(12) CWO_DECL_LAUNCH(13)
#undef CWO_DECL_LAUNCH
typedef cudaError_t (*linefft_launcher_t)(cudaStream_t s, const LineFftParams& p);

// tables.cu
cudaError_t build_twiddles(float2* tw, int n, cudaStream_t s);                 // exp(-i 2 pi m/n), fp64 -> fp32
cudaError_t build_twiddles_f64(double2* tw, int n, cudaStream_t s);            // same, kept in fp64, m < n/2
// Fresnel: spectrum of the sampled 1-D chirp, C[k] = coef * sum_{d=-N}^{N-1} exp(i pi (d pitch)^2/(lambda z)) exp(-i 2 pi dk/M)
// for two axes in one launch.  scratch: 2*M double2 per axis.
// out: C[k], k < M (2-D path); out_pairs: (re C[2j], re C[2j+1], im C[2j], im C[2j+1]), j < M/2 (separable path).
struct ChirpAxis { float2* out; float4* out_pairs; double2* scratch; const double2* tw64; int logm; double a_cycles; double2 coef; };
cudaError_t build_chirp_spectrum(const ChirpAxis& ax0, const ChirpAxis& ax1, cudaStream_t s);
// ASM split path: theta_x[k] = frac(c0 - ax ks^2 + ox ks), theta_y[l] = frac(-ay ls^2 + oy ls) (cycles, fp64 -> fp32) for
// n_planes distances at once; plane i uses tab + i*(mx+my): [theta_x (mx) | theta_y (my)].
struct AsmPlane { double c0, ax, ay, kz, ox, oy; };        // kz = z/lambda (-> resc[plane]); ox, oy: ramp, cycles per bin
constexpr int ASM_PLANE_BATCH = 128;                      // planes per launch (passed by value)
struct AsmPlaneBatch { AsmPlane p[ASM_PLANE_BATCH]; };
cudaError_t build_asm_phase_tables(float* tab, float* resc, const AsmPlaneBatch& planes, int n_planes, int mx, int my,
                                   cudaStream_t s, bool early);    // resc (may be null): z/lambda of every plane;
                                                                   // early: tab is plan-owned (may be written before the
                                                                   // preceding kernel of the stream has finished)
// t[i] = scale (-1)^(alt i) exp(i 2 pi (c0 + c1 m + c2 m^2)), m = i - n/2, i < n; up to 4 tables per launch
struct QuadTab { float2* out; int n; int alt; double c0, c1, c2, scale; };
struct QuadTabBatch { QuadTab t[4]; };
cudaError_t build_quad_phase_tables(const QuadTabBatch& b, int n_tabs, cudaStream_t s);
// out[c][r] = in[r][c] (transpose.cu); rows, cols multiples of 32
cudaError_t launch_transpose_c64(const float2* in, float2* out, int rows, int cols, cudaStream_t s);
cudaError_t launch_transpose_f32(const float* in, float* out, int rows, int cols, cudaStream_t s);
cudaError_t launch_transpose_real(const float2* in, float* out, int rows, int cols, int real_mode, cudaStream_t s);   // out[c][r] = real field of in[r][c]

// outputs.cu: Scale (Eq.(21)) and the point-light-source CGH (Eq.(23))
cudaError_t launch_minmax(const float* in, size_t n, unsigned* mm, int n_sm, cudaStream_t s);     // mm: {min, max} encoded
cudaError_t launch_scale(const float* in, float* out, size_t n, const unsigned* mm, int n_sm, cudaStream_t s);
cudaError_t launch_pls_cgh(const double* pts, int npts, float* out, int nx, int ny, double px, double py, double lambda,
                           cudaStream_t s);

}  // namespace cwo
