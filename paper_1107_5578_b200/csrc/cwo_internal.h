// cwo_internal.h -- pass descriptors and launcher declarations shared by the translation units
// of libcwo.so.  Not part of the public ABI (see include/cwo.h).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stddef.h>

namespace cwo {

enum InMode { IN_COMPLEX = 0, IN_AMP_PHASE = 1 };
enum OutMode { OUT_COMPLEX = 0, OUT_PHASOR_AMP = 1, OUT_PHASE = 2 };
enum MidMode { MID_NONE = 0, MID_TABLES = 1, MID_ASM_SPLIT = 2, MID_ASM_F64 = 3 };

struct PassParams {
    CUtensorMap tmap;         // pipelined row passes: the column-tiled workspace as a 2-D tensor (see encode_ws_tmap)
    int use_tmap;             // 1: tmap is valid, the row pass moves its workspace side with TMA tensor copies
    int use_cluster;          // 1: 16384-point forward row pass on 4-CTA clusters (cluster_kernel.cuh); tmap has 4-row boxes
    int use_fold;             // 1: 8192-point inverse row pass on one-row tiles (fold_kernel.cuh); tmap has one-row boxes
    const float2* in;
    float2* out;              // OUT_PHASE: float*
    const float* in_amp;      // IN_AMP_PHASE: amplitude [rows][pitch]
    const float* in_phase;    //               phase
    const float* out_amp;     // OUT_PHASOR_AMP: amplitude of the next plane
    int in_mode, out_mode;
    int rows;                 // row passes: number of field rows (lanes beyond it are masked)
    int pitch;                // row passes: row pitch (elements) of the row-major field and real arrays
    int ly;                   // rows kept in the column-tiled workspace
    int logwc;                // row passes: log2 of the column-tile width of the workspace
    int n_tiles;              // pipelined passes: total number of tiles (the grid is one CTA per SM)
    // batched planes (depth stack, pipelined kernels only): tile t belongs to plane t / tiles_per_plane
    int n_planes;             // 0 or 1: a single plane
    int tiles_per_plane;
    size_t in_plane_stride;   // complex elements between the planes of `in` (0: every plane reads the same data)
    size_t out_plane_stride;  // same for `out`
    int tab_plane_stride;     // MID_ASM_SPLIT: floats between the planes' [theta_x | theta_y] tables
    const float* plane_resc;  // MID_ASM_SPLIT: res_c (= z/lambda) of every plane
    int dbg;                  // CWO_OPT_EXPERIMENT bit mask (pipelined kernels): 1 no global stores, 4 no global loads
    int use_pipe;             // 1: use the pipelined form where it exists (CWO_OPT_PIPELINE)
    const float2* tw;         // forward twiddles exp(-i 2 pi m/n), m < n
    float out_scale;          // ROW_INV store
    // Mid (transfer function / impulse-response spectrum, S2/S5/S7); lane = x bin, point = y bin
    double z, inv_lam2, df_lane, df_point;   // MID_ASM_F64
    int n_lane_bins;                          // Mx (signed-bin map of the lane index)
    const float2* tab_lane;   // MID_TABLES: Cx[k] (float2);  MID_ASM_SPLIT: theta_x[k] (float, cycles)
    const float2* tab_point;  // MID_TABLES: Cy[l];           MID_ASM_SPLIT: theta_y[l]
    float res_a, res_b, res_c;  // MID_ASM_SPLIT: lambda^2 dfx^2, lambda^2 dfy^2, z/lambda
};

constexpr int MIN_LOGN = 5, MAX_LOGN = 14;

// one launcher per transform length, defined in pass_inst.cu compiled with -DCWO_LOGN=<k>
typedef cudaError_t (*pass_launcher_t)(int kind, int pad, int mid, int n_tiles, cudaStream_t s, const PassParams& p);
#define CWO_DECL_LAUNCH(k) \
    cudaError_t launch_pass_##k(int kind, int pad, int mid, int n_tiles, cudaStream_t s, const PassParams& p);
CWO_DECL_LAUNCH(5) CWO_DECL_LAUNCH(6) CWO_DECL_LAUNCH(7) CWO_DECL_LAUNCH(8) CWO_DECL_LAUNCH(9)
CWO_DECL_LAUNCH(10) CWO_DECL_LAUNCH(11) CWO_DECL_LAUNCH(12) CWO_DECL_LAUNCH(13) CWO_DECL_LAUNCH(14)
#undef CWO_DECL_LAUNCH

// tables.cu
cudaError_t build_twiddles(float2* tw, int n, cudaStream_t s);                 // exp(-i 2 pi m/n), fp64 -> fp32
cudaError_t build_twiddles_f64(double2* tw, int n, cudaStream_t s);            // same, kept in fp64, m < n/2
// Fresnel: spectrum of the sampled 1-D chirp, C[k] = coef * sum_{d=-N}^{N-1} exp(i pi (d pitch)^2/(lambda z)) exp(-i 2 pi dk/M)
// for two axes in one launch.  scratch: 2*M double2 per axis.
struct ChirpAxis { float2* out; double2* scratch; const double2* tw64; int logm; double a_cycles; double2 coef; };
cudaError_t build_chirp_spectrum(const ChirpAxis& ax0, const ChirpAxis& ax1, cudaStream_t s);
// ASM split path: theta_x[k] = frac(c0 - ax ks^2), theta_y[l] = frac(-ay ls^2) (cycles, fp64 -> fp32) for
// n_planes distances at once; plane i uses tab + i*(mx+my): [theta_x (mx) | theta_y (my)].
struct AsmPlane { double c0, ax, ay; };
constexpr int ASM_PLANE_BATCH = 128;                      // planes per launch (passed by value)
struct AsmPlaneBatch { AsmPlane p[ASM_PLANE_BATCH]; };
cudaError_t build_asm_phase_tables(float* tab, const AsmPlaneBatch& planes, int n_planes, int mx, int my, cudaStream_t s);

}  // namespace cwo
