// cwo.cu -- the C ABI of libcwo.so (include/cwo.h): plan object, argument checks, and the
// sequencing of the streaming passes that make up each call.  All arithmetic on field data
// happens in the kernels of pass_kernel.cuh / tables.cu; nothing here touches field values.
#include <math.h>
#include <new>
#include <stdint.h>
#include <string.h>

#include "../../include/cwo.h"
#include "cwo_internal.h"

using namespace cwo;

struct cwo_plan_s {
    int Nx, Ny, lognx, logny;
    double px, py, lambda;
    cudaStream_t stream;
    void* ws;
    size_t ws_bytes;
    int gs_method;
    int last_cuda_error;
    long long launches;
    float2* tw[MAX_LOGN + 2];       // fp32 twiddles per log2 length (lazily built)
    double2* tw64[MAX_LOGN + 2];    // fp64 twiddles for the chirp FFT
    float2* chirp[2][2];            // [set][axis] Fresnel spectra Cx, Cy (set 0: +z, 1: the other sign in GS)
    double2* chirp_scratch;         // 2 axes x 2M
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

static int launch(cwo_plan_t p, int logn, int kind, int n_tiles, const PassParams& pp) {
    CWO_CUDA(p, kLaunchers[logn](kind, n_tiles, p->stream, pp));
    p->launches++;
    return CWO_OK;
}

static int ensure_twiddles(cwo_plan_t p, int logn, bool want64) {
    const int n = 1 << logn;
    if (!p->tw[logn]) {
        CWO_CUDA(p, cudaMalloc(&p->tw[logn], sizeof(float2) * n));
        CWO_CUDA(p, build_twiddles(p->tw[logn], n, p->stream));
        p->launches++;
    }
    if (want64 && !p->tw64[logn]) {
        CWO_CUDA(p, cudaMalloc(&p->tw64[logn], sizeof(double2) * (n / 2)));
        CWO_CUDA(p, build_twiddles_f64(p->tw64[logn], n, p->stream));
        p->launches++;
    }
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
    if (!p) return CWO_EINVAL;
    memset(p, 0, sizeof(*p));
    p->Nx = Nx; p->Ny = Ny; p->lognx = lx; p->logny = ly;
    p->px = p->py = pitch; p->lambda = lambda;
    p->gs_method = CWO_GS_FRESNEL;
    int rc = CWO_OK;
    if (lx >= MIN_LOGN) rc = ensure_twiddles(p, lx, false);
    if (rc == CWO_OK && ly >= MIN_LOGN) rc = ensure_twiddles(p, ly, false);
    if (rc == CWO_OK && cudaStreamSynchronize(0) != cudaSuccess) rc = CWO_ECUDA;
    if (rc != CWO_OK) { cwo_plan_destroy(p); return rc; }
    *plan_out = p;
    return CWO_OK;
}

extern "C" int cwo_plan_destroy(cwo_plan_t p) {
    if (!p) return CWO_EINVAL;
    for (int i = 0; i < MAX_LOGN + 2; ++i) { cudaFree(p->tw[i]); cudaFree(p->tw64[i]); }
    for (int s = 0; s < 2; ++s) for (int a = 0; a < 2; ++a) cudaFree(p->chirp[s][a]);
    cudaFree(p->chirp_scratch);
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

extern "C" int cwo_plan_set_option(cwo_plan_t p, int key, int value) {
    if (!p) return CWO_EINVAL;
    if (key == CWO_OPT_GS_METHOD && (value == CWO_GS_FRESNEL || value == CWO_GS_ASM)) {
        p->gs_method = value;
        return CWO_OK;
    }
    return CWO_EINVAL;
}

static bool asm_sizes_ok(cwo_plan_t p) { return p->lognx >= MIN_LOGN && p->logny >= MIN_LOGN; }
static bool fresnel_sizes_ok(cwo_plan_t p) { return p->lognx + 1 <= MAX_LOGN && p->logny + 1 <= MAX_LOGN; }

static size_t prop_ws_bytes(cwo_plan_t p, int method) {
    const size_t f = sizeof(float2) * (size_t)p->Nx * p->Ny;
    return method == CWO_GS_ASM ? f : 2 * f;
}

extern "C" size_t cwo_plan_workspace_bytes(cwo_plan_t p, int op, int n) {
    (void)n;
    if (!p) return 0;
    const size_t f = sizeof(float2) * (size_t)p->Nx * p->Ny;
    switch (op) {
        case CWO_OP_ASM: return f;
        case CWO_OP_FRESNEL: return 2 * f;
        case CWO_OP_STACK: return 2 * f;
        case CWO_OP_GS: return f + prop_ws_bytes(p, p->gs_method);
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
    }
    return "unknown error";
}

extern "C" int cwo_last_cuda_error(cwo_plan_t p) { return p ? p->last_cuda_error : 0; }
extern "C" long long cwo_plan_launch_count(cwo_plan_t p) { return p ? p->launches : 0; }

// ---- addressing of the three passes ---------------------------------------------------------

static Addr addr_rowmajor_rows(int rb, int pitch) {
    Addr a; a.tile_stride = (long long)rb * pitch; a.lane_stride = (unsigned)pitch;
    a.sh = 0; a.hi_stride = 1; a.mask = 0; a.lo_stride = 0;
    return a;
}
// column-tiled workspace T[x / Wc][y][x % Wc], ly rows kept; seen from a row pass (lanes = rows)
static Addr addr_tiled_rows(int rb, int logwc, int ly) {
    const int wc = 1 << logwc;
    Addr a; a.tile_stride = (long long)rb * wc; a.lane_stride = (unsigned)wc;
    a.sh = logwc; a.hi_stride = (unsigned)ly * wc; a.mask = wc - 1; a.lo_stride = 1;
    return a;
}
// the same workspace seen from a column pass (lanes = columns of the tile, points = rows)
static Addr addr_tiled_cols(int logwc, int ly) {
    const int wc = 1 << logwc;
    Addr a; a.tile_stride = (long long)ly * wc; a.lane_stride = 1;
    a.sh = 0; a.hi_stride = (unsigned)wc; a.mask = 0; a.lo_stride = 0;
    return a;
}

// ---- one propagation = three passes ---------------------------------------------------------

struct PropIO {
    int in_mode; const float2* in; const float* in_amp; const float* in_phase;
    int out_mode; void* out; const float* out_amp;
};

struct Geometry { int logmx, logmy, mx, my, rb, logwc, wc; };

static Geometry geometry(cwo_plan_t p, int method) {
    Geometry g;
    const int pad = (method == CWO_GS_ASM) ? 0 : 1;
    g.logmx = p->lognx + pad; g.logmy = p->logny + pad;
    g.mx = 1 << g.logmx; g.my = 1 << g.logmy;
    g.rb = 1 << tile_logw(g.logmx);
    g.logwc = tile_logw(g.logmy); g.wc = 1 << g.logwc;
    return g;
}

static void fill_asm_mid(cwo_plan_t p, const Geometry& g, double z, PassParams& pp) {
    pp.mid_mode = MID_ASM_F64;
    pp.z = z;
    pp.inv_lam2 = 1.0 / (p->lambda * p->lambda);
    pp.df_lane = 1.0 / ((double)g.mx * p->px);
    pp.df_point = 1.0 / ((double)g.my * p->py);
    pp.n_lane_bins = g.mx;
    pp.mid_scale = (float)(1.0 / ((double)g.mx * (double)g.my));
}

// Build Cx, Cy for distance z into table set `set` (S2/S7: coefficient and 1/(MxMy) folded in).
static int build_fresnel_tables(cwo_plan_t p, const Geometry& g, double z, int set) {
    int rc;
    if ((rc = ensure_twiddles(p, g.logmx, true)) != CWO_OK) return rc;
    if ((rc = ensure_twiddles(p, g.logmy, true)) != CWO_OK) return rc;
    for (int s = 0; s < 2; ++s) {
        if (!p->chirp[s][0]) CWO_CUDA(p, cudaMalloc(&p->chirp[s][0], sizeof(float2) * g.mx));
        if (!p->chirp[s][1]) CWO_CUDA(p, cudaMalloc(&p->chirp[s][1], sizeof(float2) * g.my));
    }
    if (!p->chirp_scratch) CWO_CUDA(p, cudaMalloc(&p->chirp_scratch, sizeof(double2) * 2 * ((size_t)g.mx + g.my)));
    // c = exp(i 2 pi z/lambda)/(i lambda z) * px py / (Mx My), split as cx = c/sqrt|c|, cy = sqrt|c|
    const double kz = z / p->lambda, fr = kz - floor(kz);
    const double cr = cos(2.0 * M_PI * fr), ci = sin(2.0 * M_PI * fr);
    const double mag = p->px * p->py / (p->lambda * fabs(z)) / ((double)g.mx * (double)g.my);
    const double sg = z > 0 ? 1.0 : -1.0;
    // 1/(i lambda z) = -i/(lambda z):  (cr + i ci) * (-i sg) = sg*ci - i sg*cr
    const double c_re = sg * ci * mag, c_im = -sg * cr * mag;
    const double rt = sqrt(mag);
    ChirpAxis ax, ay;
    ax.out = p->chirp[set][0]; ax.scratch = p->chirp_scratch; ax.tw64 = p->tw64[g.logmx]; ax.logm = g.logmx;
    ax.a_cycles = p->px * p->px / (2.0 * p->lambda * z);
    ax.coef = make_double2(c_re / rt, c_im / rt);
    ay.out = p->chirp[set][1]; ay.scratch = p->chirp_scratch + 2 * (size_t)g.mx; ay.tw64 = p->tw64[g.logmy]; ay.logm = g.logmy;
    ay.a_cycles = p->py * p->py / (2.0 * p->lambda * z);
    ay.coef = make_double2(rt, 0.0);
    CWO_CUDA(p, build_chirp_spectrum(ax, &ay, p->stream));
    p->launches++;
    return CWO_OK;
}

// The three passes.  `ws` holds Ny rows x Mx columns in column-tile order.  For Fresnel the
// tables of set `set` must already hold the spectra for this z.
static int run_passes(cwo_plan_t p, int method, double z, int set, const PropIO& io, float2* ws) {
    const Geometry g = geometry(p, method);
    int rc;
    if ((rc = ensure_twiddles(p, g.logmx, false)) != CWO_OK) return rc;
    if ((rc = ensure_twiddles(p, g.logmy, false)) != CWO_OK) return rc;
    PassParams pp;
    // pass R: rows of u1 (zero padded to Mx) -> FFT -> ws
    memset(&pp, 0, sizeof(pp));
    pp.in = io.in; pp.in_amp = io.in_amp; pp.in_phase = io.in_phase; pp.in_mode = io.in_mode;
    pp.out = ws; pp.out_mode = OUT_COMPLEX; pp.out_scale = 1.0f;
    pp.ain = addr_rowmajor_rows(g.rb, p->Nx); pp.aout = addr_tiled_rows(g.rb, g.logwc, p->Ny);
    pp.aux_pitch = p->Nx; pp.p_in_valid = p->Nx; pp.p_out_valid = g.mx; pp.lanes_total = p->Ny;
    pp.tw = p->tw[g.logmx];
    if ((rc = launch(p, g.logmx, KIND_FWD, (p->Ny + g.rb - 1) / g.rb, pp)) != CWO_OK) return rc;
    // pass C: columns (Ny stored rows, zero padded to My) -> FFT -> x H -> IFFT -> first Ny rows, in place
    memset(&pp, 0, sizeof(pp));
    pp.in = ws; pp.out = ws; pp.in_mode = IN_COMPLEX; pp.out_mode = OUT_COMPLEX; pp.out_scale = 1.0f;
    pp.ain = pp.aout = addr_tiled_cols(g.logwc, p->Ny);
    pp.p_in_valid = p->Ny; pp.p_out_valid = p->Ny; pp.lanes_total = g.mx;
    pp.tw = p->tw[g.logmy];
    if (method == CWO_GS_ASM) fill_asm_mid(p, g, z, pp);
    else { pp.mid_mode = MID_TABLES; pp.tab_lane = p->chirp[set][0]; pp.tab_point = p->chirp[set][1]; }
    if ((rc = launch(p, g.logmy, KIND_FUSED, g.mx / g.wc, pp)) != CWO_OK) return rc;
    // pass R': rows of ws -> IFFT -> first Nx columns -> u2 (with the GS constraint if asked)
    memset(&pp, 0, sizeof(pp));
    pp.in = ws; pp.in_mode = IN_COMPLEX;
    pp.out = (float2*)io.out; pp.out_mode = io.out_mode; pp.out_amp = io.out_amp; pp.out_scale = 1.0f;
    pp.ain = addr_tiled_rows(g.rb, g.logwc, p->Ny); pp.aout = addr_rowmajor_rows(g.rb, p->Nx);
    pp.aux_pitch = p->Nx; pp.p_in_valid = g.mx; pp.p_out_valid = p->Nx; pp.lanes_total = p->Ny;
    pp.tw = p->tw[g.logmx];
    return launch(p, g.logmx, KIND_INV, (p->Ny + g.rb - 1) / g.rb, pp);
}

static bool aligned16(const void* q) { return q && !((uintptr_t)q & 15); }

extern "C" int cwo_asm(cwo_plan_t p, const cwo_c64* u1, cwo_c64* u2, double z) {
    if (!p || !aligned16(u1) || !aligned16(u2) || !isfinite(z) || !asm_sizes_ok(p)) return CWO_EINVAL;
    if (!p->ws || p->ws_bytes < cwo_plan_workspace_bytes(p, CWO_OP_ASM, 0)) return CWO_EWORKSPACE;
    PropIO io = {IN_COMPLEX, (const float2*)u1, nullptr, nullptr, OUT_COMPLEX, u2, nullptr};
    return run_passes(p, CWO_GS_ASM, z, 0, io, (float2*)p->ws);
}

extern "C" int cwo_fresnel_conv(cwo_plan_t p, const cwo_c64* u1, cwo_c64* u2, double z) {
    if (!p || !aligned16(u1) || !aligned16(u2) || !isfinite(z) || z == 0.0 || !fresnel_sizes_ok(p)) return CWO_EINVAL;
    if (!p->ws || p->ws_bytes < cwo_plan_workspace_bytes(p, CWO_OP_FRESNEL, 0)) return CWO_EWORKSPACE;
    int rc = build_fresnel_tables(p, geometry(p, CWO_GS_FRESNEL), z, 0);
    if (rc != CWO_OK) return rc;
    PropIO io = {IN_COMPLEX, (const float2*)u1, nullptr, nullptr, OUT_COMPLEX, u2, nullptr};
    return run_passes(p, CWO_GS_FRESNEL, z, 0, io, (float2*)p->ws);
}

extern "C" int cwo_propagate_stack(cwo_plan_t p, const cwo_c64* u1, const double* zs, int n, cwo_c64* out) {
    if (!p || !aligned16(u1) || !aligned16(out) || !zs || n <= 0 || !asm_sizes_ok(p)) return CWO_EINVAL;
    for (int k = 0; k < n; ++k) if (!isfinite(zs[k])) return CWO_EINVAL;
    if (!p->ws || p->ws_bytes < cwo_plan_workspace_bytes(p, CWO_OP_STACK, n)) return CWO_EWORKSPACE;
    const Geometry g = geometry(p, CWO_GS_ASM);
    const size_t f = (size_t)p->Nx * p->Ny;
    float2* A = (float2*)p->ws;
    float2* B = A + f;
    int rc;
    PassParams pp;
    // forward FFT2 of u1 once (S9): pass R, then a forward-only column pass in place
    memset(&pp, 0, sizeof(pp));
    pp.in = (const float2*)u1; pp.out = A; pp.out_scale = 1.0f;
    pp.ain = addr_rowmajor_rows(g.rb, p->Nx); pp.aout = addr_tiled_rows(g.rb, g.logwc, p->Ny);
    pp.aux_pitch = p->Nx; pp.p_in_valid = p->Nx; pp.p_out_valid = g.mx; pp.lanes_total = p->Ny;
    pp.tw = p->tw[g.logmx];
    if ((rc = launch(p, g.logmx, KIND_FWD, (p->Ny + g.rb - 1) / g.rb, pp)) != CWO_OK) return rc;
    memset(&pp, 0, sizeof(pp));
    pp.in = A; pp.out = A; pp.out_scale = 1.0f;
    pp.ain = pp.aout = addr_tiled_cols(g.logwc, p->Ny);
    pp.p_in_valid = p->Ny; pp.p_out_valid = p->Ny; pp.lanes_total = g.mx;
    pp.tw = p->tw[g.logmy];
    if ((rc = launch(p, g.logmy, KIND_FWD, g.mx / g.wc, pp)) != CWO_OK) return rc;
    for (int k = 0; k < n; ++k) {
        // per plane: x H(z_k) and inverse column transform, then inverse row transform
        memset(&pp, 0, sizeof(pp));
        pp.in = A; pp.out = B; pp.out_scale = 1.0f;
        pp.ain = pp.aout = addr_tiled_cols(g.logwc, p->Ny);
        pp.p_in_valid = p->Ny; pp.p_out_valid = p->Ny; pp.lanes_total = g.mx;
        pp.tw = p->tw[g.logmy];
        fill_asm_mid(p, g, zs[k], pp);
        if ((rc = launch(p, g.logmy, KIND_MIDINV, g.mx / g.wc, pp)) != CWO_OK) return rc;
        memset(&pp, 0, sizeof(pp));
        pp.in = B; pp.out = (float2*)out + (size_t)k * f; pp.out_scale = 1.0f;
        pp.ain = addr_tiled_rows(g.rb, g.logwc, p->Ny); pp.aout = addr_rowmajor_rows(g.rb, p->Nx);
        pp.aux_pitch = p->Nx; pp.p_in_valid = g.mx; pp.p_out_valid = p->Nx; pp.lanes_total = p->Ny;
        pp.tw = p->tw[g.logmx];
        if ((rc = launch(p, g.logmx, KIND_INV, (p->Ny + g.rb - 1) / g.rb, pp)) != CWO_OK) return rc;
    }
    return CWO_OK;
}

extern "C" int cwo_gs(cwo_plan_t p, const float* amp_src, const float* amp_dst, double z, int iters,
                      float* phase_out) {
    if (!p || !aligned16(amp_src) || !aligned16(amp_dst) || !aligned16(phase_out) || !isfinite(z) || iters < 0)
        return CWO_EINVAL;
    const int method = p->gs_method;
    if (method == CWO_GS_ASM ? !asm_sizes_ok(p) : (!fresnel_sizes_ok(p) || z == 0.0)) return CWO_EINVAL;
    if (!p->ws || p->ws_bytes < cwo_plan_workspace_bytes(p, CWO_OP_GS, 0)) return CWO_EWORKSPACE;
    const size_t f = (size_t)p->Nx * p->Ny;
    float2* g = (float2*)p->ws;          // the constrained field between propagations (8 B/px)
    float2* ws = g + f;
    int rc;
    if (method == CWO_GS_FRESNEL) {      // set 0: P(-z), set 1: P(+z)
        const Geometry geo = geometry(p, method);
        if ((rc = build_fresnel_tables(p, geo, -z, 0)) != CWO_OK) return rc;
        if (iters > 0 && (rc = build_fresnel_tables(p, geo, +z, 1)) != CWO_OK) return rc;
    }
    // steps 1-2: G = amp_dst exp(i phi0); p = phasor(P(-z)[G]); the store already forms amp_src * p
    PropIO io = {IN_AMP_PHASE, nullptr, amp_dst, phase_out,
                 iters == 0 ? OUT_PHASE : OUT_PHASOR_AMP, iters == 0 ? (void*)phase_out : (void*)g, amp_src};
    if ((rc = run_passes(p, method, -z, 0, io, ws)) != CWO_OK) return rc;
    for (int t = 0; t < iters; ++t) {
        // G = P(+z)[amp_src p]; q = phasor(G); store amp_dst * q
        PropIO fwd = {IN_COMPLEX, g, nullptr, nullptr, OUT_PHASOR_AMP, g, amp_dst};
        if ((rc = run_passes(p, method, +z, 1, fwd, ws)) != CWO_OK) return rc;
        // p = phasor(P(-z)[amp_dst q]); store amp_src * p, or the phase after the last pass
        const bool last = (t == iters - 1);
        PropIO bwd = {IN_COMPLEX, g, nullptr, nullptr, last ? OUT_PHASE : OUT_PHASOR_AMP,
                      last ? (void*)phase_out : (void*)g, amp_src};
        if ((rc = run_passes(p, method, -z, 0, bwd, ws)) != CWO_OK) return rc;
    }
    return CWO_OK;
}
