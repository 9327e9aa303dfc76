// cwo.cu -- the C ABI of libcwo.so (include/cwo.h): plan object, argument checks, and the
// sequencing of the streaming passes that make up each call.  All arithmetic on field data
// happens in the kernels of csrc/*.cuh, tables.cu and transpose.cu; nothing here touches field values.
// Every allocation and every synchronisation happens in cwo_plan(); the propagation calls only enqueue
// (include/cwo_debug.h's timing mode excepted).
#include <math.h>
#include <new>
#include <stdint.h>
#include <string.h>
#include <stdlib.h>
#include <vector>

#include "../../include/cwo.h"
#include "../../include/cwo_debug.h"
#include "cwo_internal.h"

using namespace cwo;

struct cwo_plan_s {
    int Nx, Ny, lognx, logny;
    int device;                     // the device the plan's tables live on
    double px, py, lambda;
    double off_x, off_y;            // shifted ASM / shifted Fresnel: destination offset [m] (Eq.(19), Eq.(14))
    double p1x, p1y;                // shifted Fresnel: destination pitch [m] (0: same as the source pitch)
    float2* quad[2][2];             // [axis][pre, post] chirp / ramp tables of the Fourier-form and shifted Fresnel
    cudaStream_t stream;
    void* ws;
    size_t ws_bytes;
    int gs_method, pipeline, asm_pad2x, stack_intensity, band_limit, fresnel_2d, out_real;   // out_real: CWO_OPT_OUT_REAL value (0 complex, 1..5)
    int fresnel_gather;             // include/cwo_debug.h: -1 auto (by field size), 0 transposing form, 1 gathering form
    int last_cuda_error;
    long long launches;
    float2* tw[MAX_LOGN + 2];       // fp32 twiddles per log2 length
    double2* tw64[MAX_LOGN + 2];    // fp64 twiddles for the chirp FFT
    float2* chirp[2][2];            // [set][axis] Fresnel spectra Cx, Cy (set 0: the call's z / -z in GS, 1: +z in GS)
    float4* chirp_pairs[2][2];      // the same as planar (even bin, odd bin) pairs (separable form)
    double2* chirp_scratch;         // 2 axes x 2M
    unsigned* minmax;               // cwo_scale255: {min, max} of the field as order-preserving integers
    int* tile_counter;              // persistent line-convolution kernels: {next tile, CTAs done}, zero between launches
    float* asm_tab;                 // ASM split path, one plane: [theta_x (Mx) | theta_y (My)], M up to 2N
    // include/cwo_debug.h: one CUDA event pair around every pass kernel
    int timing;
    std::vector<cudaEvent_t>* ev;   // 2 per recorded launch
    std::vector<int>* ev_tag;       // logn*16 + kind
    size_t ev_used;
};

static int ilog2_exact(int v) {
    if (v <= 0 || (v & (v - 1))) return -1;
    int l = 0;
    while ((1 << l) < v) ++l;
    return l;
}

static int fail_cuda(cwo_plan_t p, cudaError_t e) {
    p->last_cuda_error = (int)e;
    return CWO_ECUDA;
}

#define CWO_CUDA(p, expr)                                   \
    do {                                                    \
        cudaError_t e_ = (expr);                            \
        if (e_ != cudaSuccess) return fail_cuda((p), e_);   \
    } while (0)

static const pass_launcher_t kLaunchers[MAX_LOGN + 1] = {
    nullptr, nullptr, nullptr, nullptr, nullptr,
    launch_pass_5, launch_pass_6, launch_pass_7, launch_pass_8, launch_pass_9,
    launch_pass_10, launch_pass_11, launch_pass_12, launch_pass_13, launch_pass_14};
static const linefft_launcher_t kLineFft[MAX_LOGN + 1] = {
    nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr,
    launch_linefft_8, launch_linefft_9, launch_linefft_10, launch_linefft_11, launch_linefft_12, launch_linefft_13, nullptr};
static const conv_launcher_t kConv[MAX_LOGN + 1] = {
    nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr,
    launch_conv_8, launch_conv_9, launch_conv_10, launch_conv_11, launch_conv_12, launch_conv_13, nullptr};
enum { KIND_CONV = 5, KIND_TRANSPOSE = 6, KIND_LINEFFT = 7 };

// One kernel launch `f` (returns cudaError_t), counted, and bracketed by an event pair in timing mode.
template <class F>
static int launch_tagged(cwo_plan_t p, int tag, F f) {
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (p->timing) {
        while (p->ev->size() < 2 * (p->ev_used + 1)) {
            cudaEvent_t e;
            CWO_CUDA(p, cudaEventCreate(&e));
            p->ev->push_back(e);
        }
        e0 = (*p->ev)[2 * p->ev_used]; e1 = (*p->ev)[2 * p->ev_used + 1];
        if (p->ev_tag->size() <= p->ev_used) p->ev_tag->push_back(0);
        (*p->ev_tag)[p->ev_used] = tag;
        p->ev_used++;
        CWO_CUDA(p, cudaEventRecord(e0, p->stream));
    }
    CWO_CUDA(p, f());
    if (p->timing) CWO_CUDA(p, cudaEventRecord(e1, p->stream));
    p->launches++;
    return CWO_OK;
}

static int launch(cwo_plan_t p, int logn, int kind, int pad, int mid, int n_tiles, const PassParams& pp) {
    return launch_tagged(p, logn * 16 + kind, [&] { return kLaunchers[logn](kind, pad, mid, n_tiles, p->stream, pp); });
}

static bool fresnel_sizes_ok(cwo_plan_t p) { return p->lognx + 1 <= MAX_LOGN && p->logny + 1 <= MAX_LOGN; }
static bool asm_sizes_ok(cwo_plan_t p) { return p->lognx >= MIN_LOGN && p->logny >= MIN_LOGN; }

// ---- plan -------------------------------------------------------------------------------------------------

static int plan_alloc_and_build(cwo_plan_t p) {
    // twiddles: every transform length a call on this plan can use (N and 2N per axis)
    const int lens[4] = {p->lognx, p->logny, p->lognx + 1, p->logny + 1};
    for (int i = 0; i < 4; ++i) {
        const int l = lens[i];
        if (l > MAX_LOGN || p->tw[l]) continue;
        const int n = 1 << l;
        CWO_CUDA(p, cudaMalloc(&p->tw[l], sizeof(float2) * n));
        CWO_CUDA(p, build_twiddles(p->tw[l], n, 0));
        p->launches++;
    }
    const bool pad_ok = fresnel_sizes_ok(p);
    if (pad_ok) {
        const int mx = 2 * p->Nx, my = 2 * p->Ny;
        for (int i = 2; i < 4; ++i) {
            const int l = lens[i];
            if (p->tw64[l]) continue;
            CWO_CUDA(p, cudaMalloc(&p->tw64[l], sizeof(double2) * ((size_t)1 << (l - 1))));
            CWO_CUDA(p, build_twiddles_f64(p->tw64[l], 1 << l, 0));
            p->launches++;
        }
        for (int s = 0; s < 2; ++s) {
            CWO_CUDA(p, cudaMalloc(&p->chirp[s][0], sizeof(float2) * mx));
            CWO_CUDA(p, cudaMalloc(&p->chirp[s][1], sizeof(float2) * my));
            CWO_CUDA(p, cudaMalloc(&p->chirp_pairs[s][0], sizeof(float4) * p->Nx));
            CWO_CUDA(p, cudaMalloc(&p->chirp_pairs[s][1], sizeof(float4) * p->Ny));
        }
        CWO_CUDA(p, cudaMalloc(&p->chirp_scratch, sizeof(double2) * 2 * ((size_t)mx + my)));
    }
    for (int a = 0; a < 2; ++a)
        for (int k = 0; k < 2; ++k) CWO_CUDA(p, cudaMalloc(&p->quad[a][k], sizeof(float2) * (a == 0 ? p->Nx : p->Ny)));
    CWO_CUDA(p, cudaMalloc(&p->minmax, 2 * sizeof(unsigned)));
    CWO_CUDA(p, cudaMalloc(&p->tile_counter, 2 * sizeof(int)));
    CWO_CUDA(p, cudaMemsetAsync(p->tile_counter, 0, 2 * sizeof(int), 0));
    CWO_CUDA(p, cudaMalloc(&p->asm_tab, sizeof(float) * (size_t)(pad_ok ? 2 : 1) * (p->Nx + p->Ny)));
    CWO_CUDA(p, cudaStreamSynchronize(0));
    return CWO_OK;
}

extern "C" int cwo_plan(int Nx, int Ny, double pitch, double lambda, cwo_plan_t* plan_out) {
    if (!plan_out) return CWO_EINVAL;
    *plan_out = nullptr;
    const int lx = ilog2_exact(Nx), ly = ilog2_exact(Ny);
    if (lx < 4 || ly < 4 || lx > MAX_LOGN || ly > MAX_LOGN) return CWO_EINVAL;
    if (!(pitch > 0.0) || !(lambda > 0.0) || !isfinite(pitch) || !isfinite(lambda)) return CWO_EINVAL;
    int dev = 0, major = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return CWO_ECUDA;
    if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) return CWO_ECUDA;
    if (major != 10) return CWO_EUNSUPPORTED;
    cwo_plan_t p = new (std::nothrow) cwo_plan_s;
    if (!p) return CWO_ENOMEM;
    memset(p, 0, sizeof(*p));
    p->Nx = Nx; p->Ny = Ny; p->lognx = lx; p->logny = ly; p->device = dev;
    p->px = p->py = pitch; p->lambda = lambda;
    p->gs_method = CWO_GS_FRESNEL;
    p->pipeline = 1;
    p->fresnel_gather = -1;
    p->ev = new (std::nothrow) std::vector<cudaEvent_t>();
    p->ev_tag = new (std::nothrow) std::vector<int>();
    int rc = (p->ev && p->ev_tag) ? plan_alloc_and_build(p) : CWO_ENOMEM;
    if (rc != CWO_OK) {
        if (rc == CWO_ECUDA && p->last_cuda_error == (int)cudaErrorMemoryAllocation) rc = CWO_ENOMEM;
        cwo_plan_destroy(p);
        return rc;
    }
    *plan_out = p;
    return CWO_OK;
}

extern "C" int cwo_plan_destroy(cwo_plan_t p) {
    if (!p) return CWO_EINVAL;
    for (int i = 0; i < MAX_LOGN + 2; ++i) { cudaFree(p->tw[i]); cudaFree(p->tw64[i]); }
    for (int s = 0; s < 2; ++s) for (int a = 0; a < 2; ++a) { cudaFree(p->chirp[s][a]); cudaFree(p->chirp_pairs[s][a]); }
    for (int a = 0; a < 2; ++a) for (int k = 0; k < 2; ++k) cudaFree(p->quad[a][k]);
    cudaFree(p->chirp_scratch);
    cudaFree(p->asm_tab);
    cudaFree(p->tile_counter);
    cudaFree(p->minmax);
    if (p->ev) { for (cudaEvent_t e : *p->ev) cudaEventDestroy(e); delete p->ev; }
    delete p->ev_tag;
    delete p;
    return CWO_OK;
}

extern "C" int cwo_plan_set_stream(cwo_plan_t p, void* s) {
    if (!p) return CWO_EINVAL;
    p->stream = (cudaStream_t)s;
    return CWO_OK;
}

extern "C" int cwo_plan_set_pitch_xy(cwo_plan_t p, double px, double py) {
    if (!p || !(px > 0.0) || !(py > 0.0) || !isfinite(px) || !isfinite(py)) return CWO_EINVAL;
    p->px = px; p->py = py;
    return CWO_OK;
}

extern "C" int cwo_plan_set_offset(cwo_plan_t p, double ox, double oy) {
    if (!p || !isfinite(ox) || !isfinite(oy)) return CWO_EINVAL;
    p->off_x = ox; p->off_y = oy;
    return CWO_OK;
}

extern "C" int cwo_plan_set_dst_pitch_xy(cwo_plan_t p, double p1x, double p1y) {
    if (!p || !(p1x >= 0.0) || !(p1y >= 0.0) || !isfinite(p1x) || !isfinite(p1y) || ((p1x == 0.0) != (p1y == 0.0)))
        return CWO_EINVAL;
    p->p1x = p1x; p->p1y = p1y;
    return CWO_OK;
}

extern "C" int cwo_plan_set_option(cwo_plan_t p, int key, int value) {
    if (!p) return CWO_EINVAL;
    const bool flag = (value == 0 || value == 1);
    switch (key) {
        case CWO_OPT_GS_METHOD:
            if (value != CWO_GS_FRESNEL && value != CWO_GS_ASM) return CWO_EINVAL;
            p->gs_method = value;
            return CWO_OK;
        case CWO_OPT_PIPELINE:
            if (!flag) return CWO_EINVAL;
            p->pipeline = value;
            return CWO_OK;
        case CWO_OPT_ASM_PAD2X:
            if (!flag || (value && !fresnel_sizes_ok(p))) return CWO_EINVAL;
            p->asm_pad2x = value;
            return CWO_OK;
        case CWO_OPT_STACK_INTENSITY:
            if (!flag) return CWO_EINVAL;
            p->stack_intensity = value;
            return CWO_OK;
        case CWO_OPT_ASM_BAND_LIMIT:
            if (!flag) return CWO_EINVAL;
            p->band_limit = value;
            return CWO_OK;
        case CWO_OPT_OUT_REAL:
            if (value < CWO_OUT_COMPLEX || value > CWO_OUT_PHASE) return CWO_EINVAL;
            p->out_real = value;
            return CWO_OK;
    }
    return CWO_EINVAL;
}

enum { STACK_BATCH = 64 };   // measured at c4: 16 planes per launch pair 1632 us, 32: 1579 us, 64: 1553 us

static size_t align256(size_t v) { return (v + 255) & ~(size_t)255; }
static size_t stack_table_bytes(cwo_plan_t p, int n) {      // per plane: theta_x, theta_y, z/lambda
    return align256(sizeof(float) * (size_t)n * (size_t)(p->Nx + p->Ny + 1));
}

extern "C" size_t cwo_plan_workspace_bytes(cwo_plan_t p, int op, int n) {
    if (!p) return 0;
    const size_t f = sizeof(float2) * (size_t)p->Nx * p->Ny;
    switch (op) {
        case CWO_OP_ASM: return p->asm_pad2x ? 2 * f : f;
        case CWO_OP_FRESNEL: case CWO_OP_FRESNEL_FOURIER: case CWO_OP_FRESNEL_SHIFTED: return 2 * f;
        case CWO_OP_STACK: {   // spectrum + the planes in flight (up to 64 per batch of launches, minimum 1) + tables
            const int nn = n < 1 ? 1 : n;
            const int nb = nn > STACK_BATCH ? STACK_BATCH : nn;
            return (size_t)(1 + nb) * f + stack_table_bytes(p, nn);
        }
        case CWO_OP_GS: return p->gs_method == CWO_GS_ASM ? 2 * f : 3 * f;
    }
    return 0;
}

extern "C" int cwo_plan_set_workspace(cwo_plan_t p, void* dev_ptr, size_t bytes) {
    if (!p || (dev_ptr && ((uintptr_t)dev_ptr & 255))) return CWO_EINVAL;
    p->ws = dev_ptr;
    p->ws_bytes = dev_ptr ? bytes : 0;
    return CWO_OK;
}

extern "C" const char* cwo_strerror(int code) {
    switch (code) {
        case CWO_OK: return "ok";
        case CWO_EINVAL: return "invalid argument";
        case CWO_EWORKSPACE: return "workspace missing or too small";
        case CWO_EUNSUPPORTED: return "device is not compute capability 10.x (B200)";
        case CWO_ECUDA: return "CUDA runtime error (see cwo_last_cuda_error)";
        case CWO_ENOMEM: return "out of memory while building the plan";
        case CWO_ELIMIT: return "size exceeds the fixed scratch of the no-allocation entry point (CWO_SCALE255_STATIC_MAX_N)";
    }
    return "unknown error";
}

extern "C" int cwo_last_cuda_error(cwo_plan_t p) { return p ? p->last_cuda_error : 0; }

// ---- include/cwo_debug.h -------------------------------------------------------------------------------------

extern "C" int cwo_debug_set_timing(cwo_plan_t p, int on) {
    if (!p || (on != 0 && on != 1)) return CWO_EINVAL;
    p->timing = on;
    p->ev_used = 0;
    return CWO_OK;
}
extern "C" int cwo_debug_timings(cwo_plan_t p, float* ms_out, int* tag_out, int cap) {
    if (!p || cap < 0 || (cap > 0 && !ms_out)) return CWO_EINVAL;
    CWO_CUDA(p, cudaStreamSynchronize(p->stream));
    const int n = (int)p->ev_used;
    for (int i = 0; i < n && i < cap; ++i) {
        CWO_CUDA(p, cudaEventElapsedTime(&ms_out[i], (*p->ev)[2 * i], (*p->ev)[2 * i + 1]));
        if (tag_out) tag_out[i] = (*p->ev_tag)[i];
    }
    p->ev_used = 0;
    return n;
}
extern "C" long long cwo_debug_launch_count(cwo_plan_t p) { return p ? p->launches : 0; }
extern "C" int cwo_debug_set_fresnel_2d(cwo_plan_t p, int on) {
    if (!p || (on != 0 && on != 1)) return CWO_EINVAL;
    p->fresnel_2d = on;
    return CWO_OK;
}

extern "C" int cwo_debug_set_fresnel_gather(cwo_plan_t p, int mode) {
    if (!p || mode < -1 || mode > 1) return CWO_EINVAL;
    p->fresnel_gather = mode;
    return CWO_OK;
}

// ---- geometry of a propagation ------------------------------------------------------------------

enum { ROW_FWD = 0, ROW_INV = 1, COL_FWD = 2, COL_FUSED = 3, COL_MIDINV = 4 };   // == pass_kernel.cuh

#ifndef CWO_LOGW12
#define CWO_LOGW12 1
#endif
#ifndef CWO_LOGW13
#define CWO_LOGW13 1
#endif
static int tile_logw_host(int logn) {   // == fft_core.cuh tile_logw
    return logn <= 5 ? 5 : logn <= 9 ? 4 : logn == 10 ? 3 : logn == 11 ? 2 : logn == 12 ? CWO_LOGW12 : logn == 13 ? CWO_LOGW13 : 0;
}

struct Geometry { int pad, logmx, logmy, mx, my, rb, logwc, wc; };

// pad2x: cwo_asm on the zero-expanded grid (CWO_OPT_ASM_PAD2X); the stack and GS keep the circular form
static Geometry geometry(cwo_plan_t p, int method, bool pad2x = false) {
    Geometry g;
    g.pad = (method == CWO_GS_ASM && !pad2x) ? 0 : 1;
    g.logmx = p->lognx + g.pad; g.logmy = p->logny + g.pad;
    g.mx = 1 << g.logmx; g.my = 1 << g.logmy;
    g.rb = 1 << tile_logw_host(g.logmx);          // rows per row-pass tile
    g.logwc = tile_logw_host(g.logmy); g.wc = 1 << g.logwc;   // columns per column-pass tile
    return g;
}

struct PropIO {
    int in_mode; const float2* in; const float* in_amp; const float* in_phase;
    int out_mode; void* out; const float* out_amp;
    int real_mode;            // OUT_INTENSITY: RealMode (0 = |u|^2); omitted initialisers leave it 0
};

static int check_call(cwo_plan_t p) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != p->device) return CWO_EINVAL;
    return CWO_OK;
}

// ---- transfer-function tables (S2) ----------------------------------------------------------------

// ASM: decide between the fp32 split-phase path and the per-sample fp64 path, and fill the Mid fields.
// Split path requires: no evanescent bin (s_max well below 1) and a small non-paraxial residual for
// every z of the call (fp32 evaluates it to ~1e-7 relative).
static bool asm_split_ok(cwo_plan_t p, const double* zs, int n) {
    const double fxm = 0.5 / p->px, fym = 0.5 / p->py;          // |f| <= Nyquist
    const double smax = p->lambda * p->lambda * (fxm * fxm + fym * fym);
    if (!(smax <= 0.5)) return false;
    const double r = 1.0 + sqrt(1.0 - smax);
    for (int i = 0; i < n; ++i)
        if (fabs(zs[i]) / p->lambda * smax * smax / (2.0 * r * r) > 32.0) return false;
    return true;
}

// The packed Mid evaluates the residual by its series through s^7 (pipe_kernel.cuh): allowed when the first omitted
// term, (z/lambda) 429/32768 s^8 (and the geometric tail), stays below 1e-7 cycles at the largest s of the grid.
static bool asm_poly_ok(cwo_plan_t p, const double* zs, int n) {
    const double fxm = 0.5 / p->px, fym = 0.5 / p->py;
    const double smax = p->lambda * p->lambda * (fxm * fxm + fym * fym);
    if (!(smax < 0.25)) return false;
    const double tail = 429.0 / 32768.0 * pow(smax, 8) / (1.0 - smax);
    for (int i = 0; i < n; ++i)
        if (fabs(zs[i]) / p->lambda * tail > 1e-7) return false;
    return true;
}

// tab: n planes x [theta_x (mx) | theta_y (my)]; resc (may be null): z/lambda per plane.  Tiny kernels, no allocation.
// band: the call honours CWO_OPT_ASM_BAND_LIMIT and the offset (cwo_asm only: the stack and GS pass false, as cwo.h says).
static int build_asm_tables(cwo_plan_t p, const Geometry& g, const double* zs, int n, float* tab, float* resc, bool band) {
    const double dfx = 1.0 / ((double)g.mx * p->px), dfy = 1.0 / ((double)g.my * p->py);
    const bool shifted = band;
    for (int i0 = 0; i0 < n; i0 += ASM_PLANE_BATCH) {
        AsmPlaneBatch b;
        const int m = n - i0 < ASM_PLANE_BATCH ? n - i0 : ASM_PLANE_BATCH;
        for (int i = 0; i < m; ++i) {
            const double z = zs[i0 + i], kz = z / p->lambda;
            b.p[i].c0 = kz - floor(kz);
            b.p[i].ax = z * p->lambda * dfx * dfx * 0.5;
            b.p[i].ay = z * p->lambda * dfy * dfy * 0.5;
            b.p[i].kz = kz;
            b.p[i].ox = shifted ? p->off_x * dfx : 0.0;      // Eq.(19): phase ramp 2 pi (Ox fx + Oy fy), cycles per bin
            b.p[i].oy = shifted ? p->off_y * dfy : 0.0;
        }
        CWO_CUDA(p, build_asm_phase_tables(tab + (size_t)i0 * (g.mx + g.my), resc ? resc + i0 : nullptr, b, m, g.mx, g.my,
                                           p->stream, tab == p->asm_tab));
        p->launches++;
    }
    return CWO_OK;
}

// Band limits of the shifted angular spectrum method, Eq.(18) P:L213-229 (parameters per Ref.[56] of the paper,
// DESIGN.md reading R15): a bin is kept when the phase of H_SA sampled at df is not aliased,
// |O - z f/sqrt(1/lambda^2 - f^2)| <= 1/(2 df), evaluated per axis on the axis itself.  The kept bins form an
// interval (the left side is monotone in f): signed-bin range [lo, hi], empty when lo > hi.
static bool band_keep(double f, double df, double off, double lambda, double z) {
    const double inv_lam2 = 1.0 / (lambda * lambda);
    const double w = inv_lam2 - f * f;
    if (w <= 0.0) return false;
    return fabs(off - z * f / sqrt(w)) <= 0.5 / df;
}
static void band_range(double z, double lambda, double off, double df, int m, int* lo_out, int* hi_out) {
    int lo = -m / 2, hi = m / 2 - 1;
    while (lo <= hi && !band_keep((double)lo * df, df, off, lambda, z)) ++lo;
    while (hi >= lo && !band_keep((double)hi * df, df, off, lambda, z)) --hi;
    *lo_out = lo; *hi_out = hi;
}

static void fill_asm_mid(cwo_plan_t p, const Geometry& g, double z, bool split, bool poly, const float* tab, PassParams& pp,
                         bool band) {
    const double dfx = 1.0 / ((double)g.mx * p->px), dfy = 1.0 / ((double)g.my * p->py);
    pp.n_lane_bins = g.mx;
    if (split) {
        pp.tab_lane = (const float2*)tab; pp.tab_point = (const float2*)(tab + g.mx);
        pp.res_a = (float)(p->lambda * p->lambda * dfx * dfx);
        pp.res_b = (float)(p->lambda * p->lambda * dfy * dfy);
        pp.res_c = (float)(z / p->lambda);
        pp.res_poly = poly ? 1 : 0;
    } else {
        pp.z = z; pp.inv_lam2 = 1.0 / (p->lambda * p->lambda);
        pp.df_lane = dfx; pp.df_point = dfy;
        pp.off_lane = band ? p->off_x : 0.0; pp.off_point = band ? p->off_y : 0.0;
    }
    pp.band = band ? 1 : 0;
    if (band) {
        band_range(z, p->lambda, p->off_x, dfx, g.mx, &pp.band_lane_lo, &pp.band_lane_hi);
        band_range(z, p->lambda, p->off_y, dfy, g.my, &pp.band_point_lo, &pp.band_point_hi);
    }
}

// Fresnel: Cx, Cy for distance z into table set `set` (coefficient of Eq.(1) and 1/(MxMy) folded in).
static int build_fresnel_tables(cwo_plan_t p, const Geometry& g, double z, int set, double p1x = 0.0, double p1y = 0.0) {
    // shifted Fresnel (Eq.(13)): h = exp(i pi S m^2), S = p0 p1/(lambda z); p1 = p0 is the convolution form
    if (p1x == 0.0) { p1x = p->px; p1y = p->py; }
    // c = exp(i 2 pi z/lambda)/(i lambda z) * px py / (Mx My), split as cx = c/sqrt|c|, cy = sqrt|c|
    const double kz = z / p->lambda, fr = kz - floor(kz);
    const double cr = cos(2.0 * M_PI * fr), ci = sin(2.0 * M_PI * fr);
    const double mag = p->px * p->py / (p->lambda * fabs(z)) / ((double)g.mx * (double)g.my);
    const double sg = z > 0 ? 1.0 : -1.0;
    // 1/(i lambda z) = -i/(lambda z):  (cr + i ci) * (-i sg) = sg*ci - i sg*cr
    const double c_re = sg * ci * mag, c_im = -sg * cr * mag;
    const double rt = sqrt(mag);
    ChirpAxis ax, ay;
    ax.out = p->chirp[set][0]; ax.out_pairs = p->chirp_pairs[set][0];
    ax.scratch = p->chirp_scratch; ax.tw64 = p->tw64[g.logmx]; ax.logm = g.logmx;
    ax.a_cycles = p->px * p1x / (2.0 * p->lambda * z);
    ax.coef = make_double2(c_re / rt, c_im / rt);
    ay.out = p->chirp[set][1]; ay.out_pairs = p->chirp_pairs[set][1];
    ay.scratch = p->chirp_scratch + 2 * (size_t)g.mx; ay.tw64 = p->tw64[g.logmy]; ay.logm = g.logmy;
    ay.a_cycles = p->py * p1y / (2.0 * p->lambda * z);
    ay.coef = make_double2(rt, 0.0);
    CWO_CUDA(p, build_chirp_spectrum(ax, ay, p->stream));
    p->launches += 2;                                           // two-step transform: two kernels
    return CWO_OK;
}

// ---- the passes ---------------------------------------------------------------------------------------

// The column-tiled workspace T[x/Wc][y][x%Wc] seen as a 2-D float tensor: inner dimension = one column
// group (ly rows x Wc complex, contiguous), outer dimension = the Nx/Wc column groups.  A row tile
// (W rows, every x) is a box of W*Wc complex x (up to) 256 column groups: 32..128 contiguous bytes per
// column group, which TMA scatters/gathers without occupying the SM's load/store path.
typedef CUresult (*encode_tiled_t)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                   const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                   CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static encode_tiled_t get_encode_tiled() {
    static std::atomic<encode_tiled_t> fn{nullptr};
    static std::atomic<int> tried{0};
    if (!tried.load(std::memory_order_acquire)) {
        void* f = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn.store((encode_tiled_t)f, std::memory_order_release);
        tried.store(1, std::memory_order_release);
    }
    return fn.load(std::memory_order_acquire);
}
static bool encode_ws_tmap(CUtensorMap* m, const void* ws, int ly, int mx, int logwc, int w_rows, int planes = 1) {
    encode_tiled_t enc = get_encode_tiled();
    if (!enc || (w_rows << logwc) < 2) return false;          // boxes are at least 16 bytes wide
    const int wc = 1 << logwc, groups = mx >> logwc;
    cuuint64_t dims[2] = {(cuuint64_t)ly * wc * 2, (cuuint64_t)groups * planes};   // planes stack in the outer dimension
    cuuint64_t strides[1] = {(cuuint64_t)ly * wc * 8};
    cuuint32_t box[2] = {(cuuint32_t)(w_rows * wc * 2), (cuuint32_t)(groups < 256 ? groups : 256)};
    cuuint32_t es[2] = {1, 1};
    return enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<void*>(ws), dims, strides, box, es,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

static void row_params(cwo_plan_t p, const Geometry& g, PassParams& pp) {
    memset(&pp, 0, sizeof(pp));
    pp.rows = p->Ny; pp.pitch = p->Nx; pp.ly = p->Ny; pp.logwc = g.logwc;
    pp.tw = p->tw[g.logmx]; pp.out_scale = 1.0f; pp.use_pipe = p->pipeline;
}
static void col_params(cwo_plan_t p, const Geometry& g, PassParams& pp) {
    memset(&pp, 0, sizeof(pp));
    pp.ly = p->Ny; pp.tw = p->tw[g.logmy]; pp.out_scale = 1.0f; pp.use_pipe = p->pipeline;
}

// the inverse pass over 8192-point rows of complex fields runs on one-row tiles (fold_kernel.cuh) when the
// workspace pairs columns
static bool row_fold(cwo_plan_t p, const Geometry& g, bool complex_io) {
    // 4096-point rows: the one-row form wins only for zero-expanded rows (29.3 vs 31.0 us; unpadded 60.9 vs 57.8 us)
    return p->pipeline && complex_io && (g.logmx == 13 || (g.logmx == 12 && g.pad)) && g.logwc == 1;
}
static int pass_row_fwd(cwo_plan_t p, const Geometry& g, const PropIO& io, float2* ws) {
    PassParams pp; row_params(p, g, pp);
    pp.in = io.in; pp.in_amp = io.in_amp; pp.in_phase = io.in_phase; pp.in_mode = io.in_mode; pp.out = ws;
    // 16384-point rows into a column-major workspace: four rows per cluster, 32-byte pieces (cluster_kernel.cuh)
    if (p->pipeline && io.in_mode == IN_COMPLEX && g.logmx == 14 && g.logwc == 0 && p->Ny % 4 == 0 &&
        encode_ws_tmap(&pp.tmap, ws, p->Ny, g.mx, 0, 4)) {
        pp.use_cluster = 1;
        return launch(p, g.logmx, ROW_FWD, g.pad, MID_NONE, p->Ny, pp);
    }
    pp.use_tmap = (p->pipeline && encode_ws_tmap(&pp.tmap, ws, p->Ny, g.mx, g.logwc, g.rb)) ? 1 : 0;
    return launch(p, g.logmx, ROW_FWD, g.pad, MID_NONE, (p->Ny + g.rb - 1) / g.rb, pp);
}
static int pass_row_inv(cwo_plan_t p, const Geometry& g, const PropIO& io, const float2* ws, float scale) {
    PassParams pp; row_params(p, g, pp);
    pp.in = ws; pp.out = (float2*)io.out; pp.out_mode = io.out_mode; pp.out_amp = io.out_amp; pp.out_scale = scale;
    pp.real_mode = io.real_mode;
    if (row_fold(p, g, io.out_mode == OUT_COMPLEX) && encode_ws_tmap(&pp.tmap, ws, p->Ny, g.mx, g.logwc, 1)) {
        pp.use_fold = 1;
        return launch(p, g.logmx, ROW_INV, g.pad, MID_NONE, p->Ny, pp);
    }
    pp.use_tmap = (p->pipeline && encode_ws_tmap(&pp.tmap, ws, p->Ny, g.mx, g.logwc, g.rb)) ? 1 : 0;
    return launch(p, g.logmx, ROW_INV, g.pad, MID_NONE, (p->Ny + g.rb - 1) / g.rb, pp);
}

// One propagation of the two-dimensional form = pass R, pass C (fused), pass R'.  `ws` holds Ny rows x Mx columns
// in column-tile order.  Fresnel: table set `set` must hold the spectra for this z.  ASM: tables (if split) in asm_tab.
static int run_passes(cwo_plan_t p, int method, double z, int set, bool split, bool poly, const PropIO& io, float2* ws,
                      bool pad2x = false, bool band = false) {
    const Geometry g = geometry(p, method, pad2x);
    int rc;
    if ((rc = pass_row_fwd(p, g, io, ws)) != CWO_OK) return rc;
    PassParams pp; col_params(p, g, pp);
    pp.in = ws; pp.out = ws;
    int mid;
    float scale = 1.0f;
    if (method == CWO_GS_ASM) {
        mid = split ? MID_ASM_SPLIT : MID_ASM_F64;
        fill_asm_mid(p, g, z, split, poly, p->asm_tab, pp, band);
        scale = (float)(1.0 / ((double)g.mx * (double)g.my));       // 1/(MxMy) of the inverse FFT (reading R3)
    } else {
        mid = MID_TABLES; pp.tab_lane = p->chirp[set][0]; pp.tab_point = p->chirp[set][1]; pp.n_lane_bins = g.mx;
    }
    const int n_tiles = g.mx / g.wc;
    // (a persistent form of this pass with its tables in shared memory was built and measured: 101 vs 88 us at
    // 4096^2, 549 vs 520 us at 8192^2 -- static tile assignment cannot follow the SM-to-SM spread)
    rc = launch(p, g.logmy, COL_FUSED, g.pad, mid, n_tiles, pp);
    if (rc != CWO_OK) return rc;
    return pass_row_inv(p, g, io, ws, scale);
}

// CWO_OPT_OUT_REAL value -> RealMode of the stores
static int real_mode_of(cwo_plan_t p) { return p->out_real == CWO_OUT_PHASE ? REAL_PHASE : p->out_real > 0 ? p->out_real - 1 : 0; }
// output mode of the inverse row pass of the two-dimensional forms (the phase has its own store mode: GS uses it)
static int out_mode_of(cwo_plan_t p) {
    return !p->out_real ? OUT_COMPLEX : p->out_real == CWO_OUT_PHASE ? OUT_PHASE : OUT_INTENSITY;
}
static bool aligned16(const void* q) { return q && !((uintptr_t)q & 15); }

// Aliasing rules of cwo.h, checked on the pointer ranges alone (no kernel work): an output may coincide EXACTLY with the
// input it replaces (in place); any other overlap between an output and an input, or between a field and the
// workspace, is refused with CWO_EINVAL.
static bool overlaps(const void* a, size_t na, const void* b, size_t nb) {
    const uintptr_t x = (uintptr_t)a, y = (uintptr_t)b;
    return x < y + nb && y < x + na;
}
static bool partial_overlap(const void* in, const void* out, size_t n) { return in != out && overlaps(in, n, out, n); }
static bool touches_ws(cwo_plan_t p, const void* q, size_t n) { return p->ws && overlaps(q, n, p->ws, p->ws_bytes); }
// u1 -> u2, both complex Nx x Ny fields
static bool fields_alias_badly(cwo_plan_t p, const void* u1, const void* u2) {
    const size_t fb = sizeof(float2) * (size_t)p->Nx * p->Ny;
    const size_t ob = p->out_real ? fb / 2 : fb;                       // CWO_OPT_OUT_REAL: u2 holds floats
    return (u1 != u2 && overlaps(u1, fb, u2, ob)) || touches_ws(p, u1, fb) || touches_ws(p, u2, ob);
}

extern "C" int cwo_asm(cwo_plan_t p, const cwo_c64* u1, cwo_c64* u2, double z) {
    if (!p || !aligned16(u1) || !aligned16(u2) || !isfinite(z) || !asm_sizes_ok(p)) return CWO_EINVAL;
    if (check_call(p) != CWO_OK) return CWO_EINVAL;
    if (!p->ws || p->ws_bytes < cwo_plan_workspace_bytes(p, CWO_OP_ASM, 0)) return CWO_EWORKSPACE;
    if (fields_alias_badly(p, u1, u2)) return CWO_EINVAL;
    const bool pad2x = p->asm_pad2x != 0;
    const Geometry g = geometry(p, CWO_GS_ASM, pad2x);
    const bool split = asm_split_ok(p, &z, 1), poly = split && asm_poly_ok(p, &z, 1);
    int rc;
    const bool band = p->band_limit != 0;
    if (split && (rc = build_asm_tables(p, g, &z, 1, p->asm_tab, nullptr, band)) != CWO_OK) return rc;
    PropIO io = {IN_COMPLEX, (const float2*)u1, nullptr, nullptr, out_mode_of(p), u2, nullptr, real_mode_of(p)};
    return run_passes(p, CWO_GS_ASM, z, 0, split, poly, io, (float2*)p->ws, pad2x, band);
}

// ---- Fresnel diffraction, separable form (lineconv_kernel.cuh) --------------------------------------------------

static bool fresnel_separable(cwo_plan_t p) {
    return !p->fresnel_2d && p->lognx >= MIN_PAIR_LOGN && p->lognx <= MAX_PAIR_LOGN && p->logny >= MIN_PAIR_LOGN &&
           p->logny <= MAX_PAIR_LOGN;
}
// Fields that stay in L2 (<= 32 MB) skip the transposes: every pass gathers its lines from the COLUMNS of its input
// (lineconv_kernel.cuh GATHER) and writes them contiguously, i.e. in the transposed layout.  Measured: c2 42.3 -> 37.7 us,
// 2048^2 110 -> 104 us; from HBM the 8-byte gathers cost more than the transposes they replace (4096^2: 384 -> 436 us,
// 8192^2: 2043 -> 2946 us, c5 75.6 -> 94.2 ms), so larger fields keep the transposing form.
static bool separable_gather(cwo_plan_t p) {
    return p->fresnel_gather < 0 ? (size_t)p->Nx * p->Ny <= ((size_t)1 << 22) : p->fresnel_gather != 0;
}
// axis 0: convolve along x (lines = rows of a [Ny][Nx] field); axis 1: along y (lines = rows of the transposed field)
static int conv_pass(cwo_plan_t p, int axis, int variant, ConvParams& cp) {
    const int logn = axis == 0 ? p->lognx : p->logny;
    cp.tw = p->tw[logn]; cp.tw2 = p->tw[logn + 1];
    cp.n_lines = axis == 0 ? p->Ny : p->Nx;
    cp.counter = p->tile_counter;
    // (8192-point lines as four 4096-point lanes on two independent 256-thread groups of the CTA were built and
    // measured: 799 vs 830 us for one convolution, 1643 vs 1614 us for two fused -- no gain, not kept)
    return launch_tagged(p, logn * 16 + KIND_CONV, [&] { return kConv[logn](variant, p->stream, cp); });
}
static int transpose_c64(cwo_plan_t p, const float2* in, float2* out, int rows, int cols) {
    return launch_tagged(p, KIND_TRANSPOSE, [&] { return launch_transpose_c64(in, out, rows, cols, p->stream); });
}
static int transpose_f32(cwo_plan_t p, const float* in, float* out, int rows, int cols) {
    return launch_tagged(p, KIND_TRANSPOSE, [&] { return launch_transpose_f32(in, out, rows, cols, p->stream); });
}
// the last transposition of a separable call: complex u2, or a real field of it with CWO_OPT_OUT_REAL
static int transpose_out(cwo_plan_t p, const float2* in, void* u2, int rows, int cols) {
    if (!p->out_real) return transpose_c64(p, in, (float2*)u2, rows, cols);
    return launch_tagged(p, KIND_TRANSPOSE, [&] {
        return launch_transpose_real(in, (float*)u2, rows, cols, real_mode_of(p), p->stream); });
}

extern "C" int cwo_fresnel_conv(cwo_plan_t p, const cwo_c64* u1, cwo_c64* u2, double z) {
    if (!p || !aligned16(u1) || !aligned16(u2) || !isfinite(z) || z == 0.0 || !fresnel_sizes_ok(p)) return CWO_EINVAL;
    if (check_call(p) != CWO_OK) return CWO_EINVAL;
    if (!p->ws || p->ws_bytes < cwo_plan_workspace_bytes(p, CWO_OP_FRESNEL, 0)) return CWO_EWORKSPACE;
    if (fields_alias_badly(p, u1, u2)) return CWO_EINVAL;
    int rc = build_fresnel_tables(p, geometry(p, CWO_GS_FRESNEL), z, 0);
    if (rc != CWO_OK) return rc;
    // (the intensity output is formed by the last transposition: the gathering form has none)
    if (fresnel_separable(p) && separable_gather(p) && !p->out_real) {
        // y first (lines = columns of u1, gathered; result in the transposed layout [Nx][Ny]), then x (lines = columns
        // of that, gathered; result row-major [Ny][Nx])
        float2* w0 = (float2*)p->ws;
        ConvParams cp; memset(&cp, 0, sizeof(cp));
        cp.in = (const float2*)u1; cp.gather = 1; cp.in_stride = p->Nx; cp.out = w0;
        cp.tab[0] = (const ulonglong2*)p->chirp_pairs[0][1];
        if ((rc = conv_pass(p, 1, 0, cp)) != CWO_OK) return rc;                     // columns: u1 -> w0 [Nx][Ny]
        memset(&cp, 0, sizeof(cp));
        cp.in = w0; cp.gather = 1; cp.in_stride = p->Ny; cp.out = u2;
        cp.tab[0] = (const ulonglong2*)p->chirp_pairs[0][0];
        return conv_pass(p, 0, 0, cp);                                               // rows: w0 -> u2 [Ny][Nx]
    }
    if (fresnel_separable(p)) {
        const size_t f = (size_t)p->Nx * p->Ny;
        float2* w0 = (float2*)p->ws;
        float2* w1 = w0 + f;
        ConvParams cp; memset(&cp, 0, sizeof(cp));
        cp.in = (const float2*)u1; cp.out = w0; cp.tab[0] = (const ulonglong2*)p->chirp_pairs[0][0];
        if ((rc = conv_pass(p, 0, 0, cp)) != CWO_OK) return rc;                     // rows: u1 -> w0
        if ((rc = transpose_c64(p, w0, w1, p->Ny, p->Nx)) != CWO_OK) return rc;      // w1 = w0^T  [Nx][Ny]
        memset(&cp, 0, sizeof(cp));
        cp.in = w1; cp.out = w1; cp.tab[0] = (const ulonglong2*)p->chirp_pairs[0][1];
        if ((rc = conv_pass(p, 1, 0, cp)) != CWO_OK) return rc;                     // columns, in place
        return transpose_out(p, w1, u2, p->Nx, p->Ny);                               // u2 = w1^T (or |w1^T|^2)
    }
    PropIO io = {IN_COMPLEX, (const float2*)u1, nullptr, nullptr, out_mode_of(p), u2, nullptr, real_mode_of(p)};
    return run_passes(p, CWO_GS_FRESNEL, z, 0, false, false, io, (float2*)p->ws);
}

// ---- Fresnel diffraction on another destination grid: Fourier form (f2) and shifted Fresnel (f3) -------------------

static int build_quad(cwo_plan_t p, const QuadTabBatch& b) {
    CWO_CUDA(p, build_quad_phase_tables(b, 4, p->stream));
    p->launches++;
    return CWO_OK;
}
// coefficient of Eq.(1)/(9)/(11), exp(i 2 pi z/lambda)/(i lambda z) px py, as (phase in cycles, magnitude)
static void fresnel_coef(cwo_plan_t p, double z, double* cycles, double* mag) {
    const double kz = z / p->lambda;
    *cycles = (kz - floor(kz)) - (z > 0 ? 0.25 : -0.25);        // 1/(i z) = -i/z
    *mag = p->px * p->py / (p->lambda * fabs(z));
}

extern "C" int cwo_fresnel_fourier(cwo_plan_t p, const cwo_c64* u1, cwo_c64* u2, double z) {
    if (!p || !aligned16(u1) || !aligned16(u2) || !isfinite(z) || z == 0.0 || !fresnel_separable(p)) return CWO_EINVAL;
    if (check_call(p) != CWO_OK) return CWO_EINVAL;
    if (!p->ws || p->ws_bytes < cwo_plan_workspace_bytes(p, CWO_OP_FRESNEL_FOURIER, 0)) return CWO_EWORKSPACE;
    if (fields_alias_badly(p, u1, u2)) return CWO_EINVAL;
    // Eq.(8): pre = (-1)^j exp(i pi x1^2/(lambda z)); Eq.(9): post = (-1)^j exp(i pi x2^2/(lambda z)) [x c on the x axis],
    // x2 = m lambda|z|/(N p) (reading R17)
    double cc, cm; fresnel_coef(p, z, &cc, &cm);
    const double lz = p->lambda * z;
    const double p2x = p->lambda * fabs(z) / (p->Nx * p->px), p2y = p->lambda * fabs(z) / (p->Ny * p->py);
    QuadTabBatch b;
    b.t[0] = QuadTab{p->quad[0][0], p->Nx, 1, 0.0, 0.0, p->px * p->px / (2.0 * lz), 1.0};
    b.t[1] = QuadTab{p->quad[0][1], p->Nx, 1, cc, 0.0, p2x * p2x / (2.0 * lz), cm};
    b.t[2] = QuadTab{p->quad[1][0], p->Ny, 1, 0.0, 0.0, p->py * p->py / (2.0 * lz), 1.0};
    b.t[3] = QuadTab{p->quad[1][1], p->Ny, 1, 0.0, 0.0, p2y * p2y / (2.0 * lz), 1.0};
    int rc = build_quad(p, b);
    if (rc != CWO_OK) return rc;
    const size_t f = (size_t)p->Nx * p->Ny;
    float2* w0 = (float2*)p->ws;
    float2* w1 = w0 + f;
    LineFftParams lp; memset(&lp, 0, sizeof(lp));
    lp.in = (const float2*)u1; lp.out = w0; lp.pre = p->quad[0][0]; lp.post = p->quad[0][1];
    lp.tw = p->tw[p->lognx]; lp.n_lines = p->Ny; lp.inverse = z < 0;
    rc = launch_tagged(p, p->lognx * 16 + KIND_LINEFFT, [&] { return kLineFft[p->lognx](p->stream, lp); });   // rows: u1 -> w0
    if (rc != CWO_OK) return rc;
    if ((rc = transpose_c64(p, w0, w1, p->Ny, p->Nx)) != CWO_OK) return rc;
    lp.in = w1; lp.out = w1; lp.pre = p->quad[1][0]; lp.post = p->quad[1][1];
    lp.tw = p->tw[p->logny]; lp.n_lines = p->Nx;
    rc = launch_tagged(p, p->logny * 16 + KIND_LINEFFT, [&] { return kLineFft[p->logny](p->stream, lp); });   // columns, in place
    if (rc != CWO_OK) return rc;
    return transpose_out(p, w1, u2, p->Nx, p->Ny);
}

extern "C" int cwo_fresnel_shifted(cwo_plan_t p, const cwo_c64* u1, cwo_c64* u2, double z) {
    if (!p || !aligned16(u1) || !aligned16(u2) || !isfinite(z) || z == 0.0 || !fresnel_separable(p)) return CWO_EINVAL;
    if (check_call(p) != CWO_OK) return CWO_EINVAL;
    if (!p->ws || p->ws_bytes < cwo_plan_workspace_bytes(p, CWO_OP_FRESNEL_SHIFTED, 0)) return CWO_EWORKSPACE;
    if (fields_alias_badly(p, u1, u2)) return CWO_EINVAL;
    const double p1x = p->p1x > 0.0 ? p->p1x : p->px, p1y = p->p1y > 0.0 ? p->p1y : p->py;
    // spectra of h = exp(i pi S m^2) with the coefficient folded in (Eq.(13), Eq.(11))
    int rc = build_fresnel_tables(p, geometry(p, CWO_GS_FRESNEL), z, 0, p1x, p1y);
    if (rc != CWO_OK) return rc;
    // Eq.(12) and Eq.(11) with O0 = 0, O1 = (off_x, off_y) in metres (reading R16), in cycles:
    //   pre(m0)  = m0^2 p0 (p0 - p1)/(2 lambda z) - m0 p0 O1/(lambda z)
    //   post(m1) = m1^2 p1 (p1 - p0)/(2 lambda z) + m1 p1 O1/(lambda z) + O1^2/(2 lambda z)
    const double lz = p->lambda * z;
    QuadTabBatch b;
    b.t[0] = QuadTab{p->quad[0][0], p->Nx, 0, 0.0, -p->px * p->off_x / lz, p->px * (p->px - p1x) / (2.0 * lz), 1.0};
    b.t[1] = QuadTab{p->quad[0][1], p->Nx, 0, p->off_x * p->off_x / (2.0 * lz), p1x * p->off_x / lz, p1x * (p1x - p->px) / (2.0 * lz), 1.0};
    b.t[2] = QuadTab{p->quad[1][0], p->Ny, 0, 0.0, -p->py * p->off_y / lz, p->py * (p->py - p1y) / (2.0 * lz), 1.0};
    b.t[3] = QuadTab{p->quad[1][1], p->Ny, 0, p->off_y * p->off_y / (2.0 * lz), p1y * p->off_y / lz, p1y * (p1y - p->py) / (2.0 * lz), 1.0};
    if ((rc = build_quad(p, b)) != CWO_OK) return rc;
    if (separable_gather(p) && !p->out_real) {
        float2* w0 = (float2*)p->ws;
        ConvParams cp; memset(&cp, 0, sizeof(cp));
        cp.in = (const float2*)u1; cp.gather = 1; cp.in_stride = p->Nx; cp.out = w0;
        cp.tab[0] = (const ulonglong2*)p->chirp_pairs[0][1]; cp.pre = p->quad[1][0]; cp.post = p->quad[1][1];
        if ((rc = conv_pass(p, 1, 4, cp)) != CWO_OK) return rc;                     // y: u1 -> w0 [Nx][Ny]
        memset(&cp, 0, sizeof(cp));
        cp.in = w0; cp.gather = 1; cp.in_stride = p->Ny; cp.out = u2;
        cp.tab[0] = (const ulonglong2*)p->chirp_pairs[0][0]; cp.pre = p->quad[0][0]; cp.post = p->quad[0][1];
        return conv_pass(p, 0, 4, cp);                                               // x: w0 -> u2 [Ny][Nx]
    }
    const size_t f = (size_t)p->Nx * p->Ny;
    float2* w0 = (float2*)p->ws;
    float2* w1 = w0 + f;
    ConvParams cp; memset(&cp, 0, sizeof(cp));
    cp.in = (const float2*)u1; cp.out = w0; cp.tab[0] = (const ulonglong2*)p->chirp_pairs[0][0];
    cp.pre = p->quad[0][0]; cp.post = p->quad[0][1];
    if ((rc = conv_pass(p, 0, 4, cp)) != CWO_OK) return rc;
    if ((rc = transpose_c64(p, w0, w1, p->Ny, p->Nx)) != CWO_OK) return rc;
    memset(&cp, 0, sizeof(cp));
    cp.in = w1; cp.out = w1; cp.tab[0] = (const ulonglong2*)p->chirp_pairs[0][1];
    cp.pre = p->quad[1][0]; cp.post = p->quad[1][1];
    if ((rc = conv_pass(p, 1, 4, cp)) != CWO_OK) return rc;
    return transpose_out(p, w1, u2, p->Nx, p->Ny);
}

// ---- output conversions (outputs.cu) ----------------------------------------------------------------------------

enum { KIND_MINMAX = 8, KIND_SCALE = 9, KIND_PLS = 10 };

extern "C" int cwo_scale255(cwo_plan_t p, const float* in, float* out, size_t n) {
    if (!p || !aligned16(in) || !aligned16(out) || n == 0) return CWO_EINVAL;
    if (partial_overlap(in, out, sizeof(float) * n)) return CWO_EINVAL;
    if (check_call(p) != CWO_OK) return CWO_EINVAL;
    DeviceInfo* d = device_info();
    if (!d) return CWO_EINVAL;
    CWO_CUDA(p, cudaMemsetAsync(p->minmax, 0xff, sizeof(unsigned), p->stream));
    CWO_CUDA(p, cudaMemsetAsync(p->minmax + 1, 0x00, sizeof(unsigned), p->stream));
    int rc = launch_tagged(p, KIND_MINMAX, [&] { return launch_minmax(in, n, p->minmax, d->n_sm, p->stream); });
    if (rc != CWO_OK) return rc;
    return launch_tagged(p, KIND_SCALE, [&] { return launch_scale(in, out, n, p->minmax, d->n_sm, p->stream); });
}

extern "C" int cwo_pls_cgh(cwo_plan_t p, const double* pts, int n, float* out) {
    if (!p || !aligned16(pts) || !aligned16(out) || n <= 0) return CWO_EINVAL;
    if (overlaps(pts, sizeof(double) * 4 * (size_t)n, out, sizeof(float) * (size_t)p->Nx * p->Ny)) return CWO_EINVAL;
    if (check_call(p) != CWO_OK) return CWO_EINVAL;
    return launch_tagged(p, KIND_PLS, [&] {
        return launch_pls_cgh(pts, n, out, p->Nx, p->Ny, p->px, p->py, p->lambda, p->stream); });
}

extern "C" int cwo_propagate_stack(cwo_plan_t p, const cwo_c64* u1, const double* zs, int n, void* out) {
    if (!p || !aligned16(u1) || !aligned16(out) || !zs || n <= 0 || !asm_sizes_ok(p)) return CWO_EINVAL;
    for (int k = 0; k < n; ++k) if (!isfinite(zs[k])) return CWO_EINVAL;
    if (check_call(p) != CWO_OK) return CWO_EINVAL;
    const Geometry g = geometry(p, CWO_GS_ASM);
    const size_t f = (size_t)p->Nx * p->Ny, fb = sizeof(float2) * f, tb = stack_table_bytes(p, n);
    if (!p->ws || p->ws_bytes < 2 * fb + tb) return CWO_EWORKSPACE;               // the minimum: one plane in flight
    {
        const size_t ob = (p->stack_intensity ? fb / 2 : fb) * (size_t)n;
        if (overlaps(u1, fb, out, ob) || touches_ws(p, u1, fb) || touches_ws(p, out, ob)) return CWO_EINVAL;
    }
    int cap = (int)((p->ws_bytes - tb) / fb) - 1;                                  // planes in flight
    if (cap > STACK_BATCH) cap = STACK_BATCH;                                      // the measured and tested batch size
    float2* A = (float2*)p->ws;       // FFT2[u1] in column-tile order, computed once (S9)
    float2* B = A + f;                // planes between their column and row pass
    float* tab = (float*)((unsigned char*)p->ws + (size_t)(1 + cap) * fb);        // n x [theta_x | theta_y], then z/lambda
    float* resc = tab + (size_t)n * (g.mx + g.my);
    const int tab_stride = g.mx + g.my;
    const bool intensity = p->stack_intensity != 0;
    const int out_mode = intensity ? OUT_INTENSITY : OUT_COMPLEX;
    const size_t out_plane = intensity ? f / 2 : f;                                // in float2 units
    int rc;
    const bool split = asm_split_ok(p, zs, n), poly = split && asm_poly_ok(p, zs, n);
    // Batched form (pipelined kernels, split-phase H): one column launch and one row launch cover as many planes
    // as the workspace holds, so the persistent CTAs fill and drain once per batch instead of once per plane.
    const bool pipe_len = g.logmx >= 10 && g.logmx <= 12 && g.logmy >= 10 && g.logmy <= 12;
    bool batched = split && p->pipeline && pipe_len && cap >= 2 && p->Ny % g.rb == 0;
    // the tensor maps of a full batch and of the remainder batch, encoded BEFORE anything is enqueued
    CUtensorMap batch_map[2];
    const int nb_full = cap < n ? cap : n, nb_rem = n % nb_full;
    if (batched)
        batched = encode_ws_tmap(&batch_map[0], B, p->Ny, g.mx, g.logwc, g.rb, nb_full) &&
                  (nb_rem == 0 || encode_ws_tmap(&batch_map[1], B, p->Ny, g.mx, g.logwc, g.rb, nb_rem));
    // the band limit and the offset are cwo_asm's (cwo.h): the band depends on |z|, and a batch shares one PassParams
    if (split && (rc = build_asm_tables(p, g, zs, n, tab, resc, false)) != CWO_OK) return rc;
    PropIO io = {IN_COMPLEX, (const float2*)u1, nullptr, nullptr, out_mode, nullptr, nullptr};
    if ((rc = pass_row_fwd(p, g, io, A)) != CWO_OK) return rc;
    PassParams pp; col_params(p, g, pp);
    pp.in = A; pp.out = A;
    if ((rc = launch(p, g.logmy, COL_FWD, 0, MID_NONE, g.mx / g.wc, pp)) != CWO_OK) return rc;
    const float scale = (float)(1.0 / ((double)g.mx * (double)g.my));
    if (batched) {
        for (int k0 = 0; k0 < n;) {
            const int nb = n - k0 < cap ? n - k0 : cap;
            col_params(p, g, pp);
            pp.in = A; pp.out = B;
            fill_asm_mid(p, g, zs[k0], true, poly, tab + (size_t)k0 * tab_stride, pp, false);
            pp.n_planes = nb; pp.tiles_per_plane = g.mx / g.wc; pp.in_plane_stride = 0; pp.out_plane_stride = f;
            pp.tab_plane_stride = tab_stride; pp.plane_resc = resc + k0;
            if ((rc = launch(p, g.logmy, COL_MIDINV, 0, MID_ASM_SPLIT, nb * (g.mx / g.wc), pp)) != CWO_OK) return rc;
            PassParams rp; row_params(p, g, rp);
            rp.in = B; rp.out = (float2*)out + (size_t)k0 * out_plane; rp.out_mode = out_mode; rp.out_scale = scale;
            rp.n_planes = nb; rp.tiles_per_plane = p->Ny / g.rb; rp.in_plane_stride = f; rp.out_plane_stride = out_plane;
            rp.tmap = batch_map[nb == nb_full ? 0 : 1]; rp.use_tmap = 1;
            if ((rc = launch(p, g.logmx, ROW_INV, 0, MID_NONE, nb * (p->Ny / g.rb), rp)) != CWO_OK) return rc;
            k0 += nb;
        }
        return CWO_OK;
    }
    for (int k = 0; k < n; ++k) {
        col_params(p, g, pp);
        pp.in = A; pp.out = B;
        fill_asm_mid(p, g, zs[k], split, poly, tab + (size_t)k * tab_stride, pp, false);
        if ((rc = launch(p, g.logmy, COL_MIDINV, 0, split ? MID_ASM_SPLIT : MID_ASM_F64, g.mx / g.wc, pp)) != CWO_OK)
            return rc;
        io.out = (float2*)out + (size_t)k * out_plane;
        if ((rc = pass_row_inv(p, g, io, B, scale)) != CWO_OK) return rc;
    }
    return CWO_OK;
}

// Gerchberg-Saxton with the separable Fresnel propagator.  Propagations P_1 = P(-z), P_2 = P(+z), P_3 = P(-z), ...;
// P_m convolves x then y for odd m and y then x for even m, so that the last convolution of P_m, the constraint and
// the first convolution of P_(m+1) act on the same lines and run as ONE pass; the field is transposed between passes.
static int gs_fresnel_separable(cwo_plan_t p, const float* amp_src, const float* amp_dst, double z, int iters,
                                float* phase_out) {
    const size_t f = (size_t)p->Nx * p->Ny;
    float2* cur = (float2*)p->ws;                 // [Ny][Nx] after x passes, [Nx][Ny] after y passes
    float2* oth = cur + f;
    float* amp_src_t = (float*)((float2*)p->ws + 2 * f);   // amp_src transposed, [Nx][Ny]
    const Geometry geo = geometry(p, CWO_GS_FRESNEL);
    int rc;
    if ((rc = build_fresnel_tables(p, geo, -z, 0)) != CWO_OK) return rc;                  // set 0: P(-z)
    if (iters > 0 && (rc = build_fresnel_tables(p, geo, +z, 1)) != CWO_OK) return rc;     // set 1: P(+z)
    const ulonglong2* X[2] = {(const ulonglong2*)p->chirp_pairs[0][0], (const ulonglong2*)p->chirp_pairs[1][0]};
    const ulonglong2* Y[2] = {(const ulonglong2*)p->chirp_pairs[0][1], (const ulonglong2*)p->chirp_pairs[1][1]};
    if (iters > 0 && (rc = transpose_f32(p, amp_src, amp_src_t, p->Ny, p->Nx)) != CWO_OK) return rc;
    ConvParams cp;
    // pass 0: G = amp_dst exp(i phi0) -> x convolution of P_1
    memset(&cp, 0, sizeof(cp));
    cp.in_amp = amp_dst; cp.in_phase = phase_out; cp.out = cur; cp.tab[0] = X[0];
    if ((rc = conv_pass(p, 0, 1, cp)) != CWO_OK) return rc;
    if (separable_gather(p)) {
        // every later pass gathers its lines from the columns of the previous pass' output: cur is [Ny][Nx] before an
        // odd (y) pass and [Nx][Ny] before an even (x) pass
        for (int m = 1; m <= 2 * iters; ++m) {
            memset(&cp, 0, sizeof(cp));
            cp.in = cur; cp.out = oth; cp.gather = 1;
            if (m & 1) { cp.tab[0] = Y[0]; cp.tab[1] = Y[1]; cp.mid_amp = amp_src_t; cp.in_stride = p->Nx; }
            else { cp.tab[0] = X[1]; cp.tab[1] = X[0]; cp.mid_amp = amp_dst; cp.in_stride = p->Ny; }
            if ((rc = conv_pass(p, (m & 1) ? 1 : 0, 2, cp)) != CWO_OK) return rc;
            float2* t = cur; cur = oth; oth = t;
        }
        memset(&cp, 0, sizeof(cp));
        cp.in = cur; cp.out = oth; cp.tab[0] = Y[0]; cp.gather = 1; cp.in_stride = p->Nx;
        if ((rc = conv_pass(p, 1, 3, cp)) != CWO_OK) return rc;
        return transpose_f32(p, (const float*)oth, phase_out, p->Nx, p->Ny);
    }
    if ((rc = transpose_c64(p, cur, oth, p->Ny, p->Nx)) != CWO_OK) return rc;
    { float2* t = cur; cur = oth; oth = t; }
    for (int m = 1; m <= 2 * iters; ++m) {
        memset(&cp, 0, sizeof(cp));
        cp.in = cur; cp.out = cur;
        if (m & 1) {   // y of P_m (-z), amplitude of the source plane, y of P_(m+1) (+z); lines = columns
            cp.tab[0] = Y[0]; cp.tab[1] = Y[1]; cp.mid_amp = amp_src_t;
            if ((rc = conv_pass(p, 1, 2, cp)) != CWO_OK) return rc;
            if ((rc = transpose_c64(p, cur, oth, p->Nx, p->Ny)) != CWO_OK) return rc;
        } else {       // x of P_m (+z), amplitude of the destination plane, x of P_(m+1) (-z); lines = rows
            cp.tab[0] = X[1]; cp.tab[1] = X[0]; cp.mid_amp = amp_dst;
            if ((rc = conv_pass(p, 0, 2, cp)) != CWO_OK) return rc;
            if ((rc = transpose_c64(p, cur, oth, p->Ny, p->Nx)) != CWO_OK) return rc;
        }
        float2* t = cur; cur = oth; oth = t;
    }
    // last pass: y of P_(2 iters + 1) (-z), phase; the result is transposed back into phase_out
    memset(&cp, 0, sizeof(cp));
    cp.in = cur; cp.out = oth; cp.tab[0] = Y[0];
    if ((rc = conv_pass(p, 1, 3, cp)) != CWO_OK) return rc;
    return transpose_f32(p, (const float*)oth, phase_out, p->Nx, p->Ny);
}

extern "C" int cwo_gs(cwo_plan_t p, const float* amp_src, const float* amp_dst, double z, int iters,
                      float* phase_out) {
    if (!p || !aligned16(amp_src) || !aligned16(amp_dst) || !aligned16(phase_out) || !isfinite(z) || iters < 0)
        return CWO_EINVAL;
    const int method = p->gs_method;
    if (method == CWO_GS_ASM ? !asm_sizes_ok(p) : (!fresnel_sizes_ok(p) || z == 0.0)) return CWO_EINVAL;
    if (check_call(p) != CWO_OK) return CWO_EINVAL;
    if (!p->ws || p->ws_bytes < cwo_plan_workspace_bytes(p, CWO_OP_GS, 0)) return CWO_EWORKSPACE;
    {   // the two amplitudes are only read (they may coincide); phase_out is written
        const size_t rb = sizeof(float) * (size_t)p->Nx * p->Ny;
        if (overlaps(amp_src, rb, phase_out, rb) || overlaps(amp_dst, rb, phase_out, rb) || touches_ws(p, amp_src, rb) ||
            touches_ws(p, amp_dst, rb) || touches_ws(p, phase_out, rb))
            return CWO_EINVAL;
    }
    if (method == CWO_GS_FRESNEL && fresnel_separable(p)) return gs_fresnel_separable(p, amp_src, amp_dst, z, iters, phase_out);
    const size_t f = (size_t)p->Nx * p->Ny;
    float2* g = (float2*)p->ws;          // the constrained field between propagations (8 B/px)
    float2* ws = g + f;
    const Geometry geo = geometry(p, method);
    int rc;
    bool split = false, poly = false;
    if (method == CWO_GS_FRESNEL) {      // set 0: P(-z), set 1: P(+z)
        if ((rc = build_fresnel_tables(p, geo, -z, 0)) != CWO_OK) return rc;
        if (iters > 0 && (rc = build_fresnel_tables(p, geo, +z, 1)) != CWO_OK) return rc;
    } else {
        split = asm_split_ok(p, &z, 1);
        poly = split && asm_poly_ok(p, &z, 1);
    }
    // The ASM tables hold one z at a time; they are rebuilt before each propagation (tiny kernel).
    auto prop = [&](double zz, int set, const PropIO& io) -> int {
        if (method == CWO_GS_ASM && split) { int r = build_asm_tables(p, geo, &zz, 1, p->asm_tab, nullptr, false); if (r != CWO_OK) return r; }
        return run_passes(p, method, zz, set, split, poly, io, ws);
    };
    // steps 1-2: G = amp_dst exp(i phi0); p = phasor(P(-z)[G]); the store already forms amp_src * p
    PropIO io = {IN_AMP_PHASE, nullptr, amp_dst, phase_out,
                 iters == 0 ? OUT_PHASE : OUT_PHASOR_AMP, iters == 0 ? (void*)phase_out : (void*)g, amp_src};
    if ((rc = prop(-z, 0, io)) != CWO_OK) return rc;
    for (int t = 0; t < iters; ++t) {
        // G = P(+z)[amp_src p]; q = phasor(G); store amp_dst * q
        PropIO fwd = {IN_COMPLEX, g, nullptr, nullptr, OUT_PHASOR_AMP, g, amp_dst};
        if ((rc = prop(+z, 1, fwd)) != CWO_OK) return rc;
        // p = phasor(P(-z)[amp_dst q]); store amp_src * p, or the phase after the last pass
        const bool last = (t == iters - 1);
        PropIO bwd = {IN_COMPLEX, g, nullptr, nullptr, last ? OUT_PHASE : OUT_PHASOR_AMP,
                      last ? (void*)phase_out : (void*)g, amp_src};
        if ((rc = prop(-z, 0, bwd)) != CWO_OK) return rc;
    }
    return CWO_OK;
}
