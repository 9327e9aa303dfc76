/*
 * cwo.h -- C ABI of libcwo.so: FFT-based scalar light propagation on one NVIDIA B200 (sm_100a).
 *
 * The calls follow the paper's statement of the problem (arxiv/paper_1107_5578, "CWO++"):
 * a source plane u1, a destination plane u2, a propagation distance z, a wavelength and the
 * sampling pitches.  P:Lnnn = line nnn of the paper text.
 *
 * Common rules
 *   Layout     Every field is a DEVICE pointer, row-major [Ny][Nx], x fastest, dense (row stride
 *              Nx), 16-byte aligned.  Complex fields are interleaved (re, im) float pairs
 *              (8*Nx*Ny bytes); real fields are float (4*Nx*Ny bytes).
 *   Ownership  The caller owns every buffer, including the workspace.  A plan owns only small
 *              lookup tables (a few MiB at most); ALL of them are allocated, built and synchronised
 *              inside cwo_plan().  No other call allocates, frees or synchronises anything.
 *   Asynchrony cwo_asm / cwo_fresnel_* / cwo_propagate_stack / cwo_gs / cwo_scale255 / cwo_pls_cgh only ENQUEUE kernels on the
 *              plan's stream and return (they may be captured into a CUDA graph); results are valid
 *              once the caller has synchronised that stream.  No host<->device copies.  Host arrays
 *              (zs) are read before return.
 *   Aliasing   u2 == u1 (exact in-place, as the paper's c.Diffract) is allowed; so is out == in for
 *              cwo_scale255.  Any other overlap of an output with an input (stack: out with u1; cwo_gs: phase_out
 *              with an amplitude; cwo_pls_cgh: out with pts), and any overlap of a field with the workspace, returns
 *              CWO_EINVAL (a check of the pointer ranges; nothing is enqueued).
 *   Errors     int return, CWO_OK == 0, negative on failure.  Nothing is enqueued when a call
 *              returns CWO_EINVAL / CWO_EWORKSPACE / CWO_EUNSUPPORTED.  No exceptions, no
 *              global state; use one plan per host thread at a time, on the device it was made on.
 *   Sizes      Nx, Ny powers of two.  cwo_asm / cwo_propagate_stack: 32..16384 per axis.
 *              cwo_fresnel_conv (transforms of 2Nx x 2Ny): 16..8192 per axis.  cwo_gs: the
 *              range of its propagator.  cwo_fresnel_fourier / cwo_fresnel_shifted: 256..8192 per axis.
 *   Sign       z < 0 is back-propagation for both methods.
 *   FFT        forward kernel exp(-i 2 pi jk/n), inverse exp(+i 2 pi jk/n) scaled 1/(Mx*My)
 *              (the paper is silent; with this choice cwo_asm at z = 0 is the identity).
 */
#ifndef CWO_H_
#define CWO_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct cwo_plan_s* cwo_plan_t;
typedef struct { float re, im; } cwo_c64;      /* == float2 == torch.complex64 element */

enum {
    CWO_OK = 0,
    CWO_EINVAL = -1,        /* bad argument: null/unaligned pointer, unsupported size, lambda/pitch <= 0,
                               non-finite z, z == 0 for Fresnel, n <= 0, iters < 0, plan used on another device */
    CWO_EWORKSPACE = -2,    /* workspace missing or smaller than cwo_plan_workspace_bytes() */
    CWO_EUNSUPPORTED = -3,  /* current device is not compute capability 10.x */
    CWO_ECUDA = -4,         /* CUDA runtime failure; code via cwo_last_cuda_error() */
    CWO_ENOMEM = -5,        /* host or device allocation failed in cwo_plan() */
    CWO_ELIMIT = -6         /* cwo_scale255_static: n exceeds CWO_SCALE255_STATIC_MAX_N (its scratch is a fixed array) */
};

enum { CWO_OP_ASM = 1, CWO_OP_FRESNEL = 2, CWO_OP_STACK = 3, CWO_OP_GS = 4, CWO_OP_FRESNEL_FOURIER = 5,
       CWO_OP_FRESNEL_SHIFTED = 6 };

enum {
    CWO_OPT_GS_METHOD = 1,  /* value: CWO_GS_FRESNEL (default; BASELINE config 5) or CWO_GS_ASM
                               (the paper's Listing 8) */
    CWO_OPT_PIPELINE = 3,   /* value 1 (default): persistent, prefetching kernels where they exist;
                               0: one CTA per tile everywhere.  Same arithmetic either way. */
    CWO_OPT_ASM_PAD2X = 5,  /* value 1: cwo_asm runs on the calculation area expanded to 2Nx x 2Ny with zeros and crops
                               (the paper's own form of the method, Table 2: no wrap-around; frequency
                               sampling 1/(2 N pitch)); needs Nx, Ny <= 8192 and a workspace of 16*Nx*Ny.  Default 0:
                               circular Nx x Ny form.  cwo_propagate_stack and cwo_gs always use the circular form. */
    CWO_OPT_STACK_INTENSITY = 6, /* value 1: cwo_propagate_stack writes the INTENSITY |u|^2 of every plane (Eq.(20),
                               P:L254-256; the quantity the paper's 3-D example renders) as float [n][Ny][Nx]
                               instead of the complex amplitude: half the output bytes.  Default 0. */
    CWO_OPT_ASM_BAND_LIMIT = 7, /* value 1: cwo_asm multiplies the transfer function by the two Rect band limits of
                               Eq.(18)-(19) for the on-axis case: bins with |fx| > 1/(lambda
                               sqrt((2 dfx z)^2 + 1)) (same in y) are zeroed, which removes the aliased part of H at
                               long distances.  Default 0.  cwo_propagate_stack and cwo_gs ignore this option and the
                               offset of cwo_plan_set_offset: they always apply the plain H of Eq.(16). */
    CWO_OPT_OUT_REAL = 8     /* value CWO_OUT_INTENSITY .. CWO_OUT_PHASE: cwo_asm, cwo_fresnel_conv, cwo_fresnel_fourier and
                               cwo_fresnel_shifted write a REAL field of u2 (section 5: the paper's Intensity(),
                               Amp, Re(), Im, Phase() applied to the diffracted plane, e.g. Diffract -> Intensity of Listing 1,
                               P:L245-252) as float [Ny][Nx] through the u2 pointer (4*Nx*Ny bytes) instead of the complex
                               amplitude: the conversion happens in the call's last store, there is no extra pass.
                               u2 == u1 stays allowed.  Default CWO_OUT_COMPLEX.  (The stack has CWO_OPT_STACK_INTENSITY.) */
};
enum { CWO_GS_FRESNEL = 0, CWO_GS_ASM = 1 };
enum { CWO_OUT_COMPLEX = 0,
       CWO_OUT_INTENSITY = 1,   /* |u2|^2, Eq.(20) */
       CWO_OUT_AMPLITUDE = 2,   /* |u2| */
       CWO_OUT_RE = 3,          /* real part, Eq.(24) */
       CWO_OUT_IM = 4,          /* imaginary part */
       CWO_OUT_PHASE = 5 };     /* atan2(im, re) in [-pi, pi], Eq.(25); 0 where u2 == 0 */

/* Plane parameters (SetPitch / SetWaveLength / Create).  pitch_x = pitch_y = pitch
 * [m], lambda [m].  Frequency sampling is 1/(M*pitch) with M the transform size.
 * Allocates and builds every table the plan will ever need on the current CUDA device (tiny kernels
 * on the null stream, synchronised before return); the plan must be used on that device. */
int cwo_plan(int Nx, int Ny, double pitch, double lambda, cwo_plan_t* plan_out);
int cwo_plan_destroy(cwo_plan_t plan);

/* Stream (a cudaStream_t passed as void*) that all later calls enqueue on.  Default: null stream. */
int cwo_plan_set_stream(cwo_plan_t plan, void* cuda_stream);

/* The paper allows px != py (SetPitch(px, py)). */
int cwo_plan_set_pitch_xy(cwo_plan_t plan, double px, double py);

int cwo_plan_set_option(cwo_plan_t plan, int key, int value);

/* Shifted angular spectrum method (Eq.(18)-(19); the paper's SetOffset): with CWO_OPT_ASM_BAND_LIMIT
 * on, cwo_asm samples the destination plane on a window displaced by (ox, oy) metres from the axis of the source
 * window: H is multiplied by the phase ramp exp(i 2 pi (ox fx + oy fy)) and the band limits follow the shift.
 * Default (0, 0): on-axis, band-limited only. */
int cwo_plan_set_offset(cwo_plan_t plan, double ox, double oy);

/* Sampling pitch of the DESTINATION plane for cwo_fresnel_shifted (Eq.(14): p_x1, p_y1) [m].
 * (0, 0) (the default) = the source pitch.  Both zero or both positive. */
int cwo_plan_set_dst_pitch_xy(cwo_plan_t plan, double p1x, double p1y);

/* Workspace a call needs, in bytes (n = number of planes for CWO_OP_STACK, ignored otherwise):
 *   ASM      8*Nx*Ny            the row-transformed field in column-tile order; needed for u2 != u1 too, because
 *                               the inverse row pass cannot write row-major rows over the column-tiled data it reads
 *            (16*Nx*Ny with CWO_OPT_ASM_PAD2X)
 *   FRESNEL  16*Nx*Ny           two copies of the field (the 2Nx x 2Ny padded array is never stored)
 *   STACK    8*Nx*Ny*(1 + min(n, 64)) + 4*n*(Nx+Ny+1) rounded up to 256
 *                               spectrum + the planes in flight between their column and row pass + the planes'
 *                               phase tables; cwo_propagate_stack accepts anything >= 16*Nx*Ny + the tables and
 *                               batches as many planes as fit
 *   FRESNEL_FOURIER, FRESNEL_SHIFTED   16*Nx*Ny
 *   GS       24*Nx*Ny (Fresnel) / 16*Nx*Ny (ASM)
 * Returns 0 for an unknown op. */
size_t cwo_plan_workspace_bytes(cwo_plan_t plan, int op, int n);

/* Device memory the calls may scribble on; 256-byte aligned; must outlive the calls using it. */
int cwo_plan_set_workspace(cwo_plan_t plan, void* dev_ptr, size_t bytes);

/* Angular spectrum method, Eq.(15)-(17):
 *   u2 = IFFT2[ FFT2[u1] * H ],  H(k,l) = exp(i 2 pi z sqrt(1/lambda^2 - fx(k)^2 - fy(l)^2)),
 *   H = 0 where the radicand is negative (evanescent), fx(k) = k_signed/(Nx*px).
 * Unpadded Nx x Ny circular transform.  z = 0 is the identity. */
int cwo_asm(cwo_plan_t plan, const cwo_c64* u1, cwo_c64* u2, double z);

/* Fresnel diffraction, convolution form, Eq.(1)-(6) with the 2Nx x 2Ny expansion of
 * P:L235:  u2 = exp(i 2 pi z/lambda)/(i lambda z) * px*py * crop( IFFT2[ FFT2[pad u1] * FFT2[h_F] ] ),
 * h_F(m,n) = exp(i pi ((m px)^2 + (n py)^2)/(lambda z)) sampled at taps -N..N-1 per axis; i.e. the
 * exact linear convolution of u1 with the sampled impulse response.  z == 0 -> CWO_EINVAL. */
int cwo_fresnel_conv(cwo_plan_t plan, const cwo_c64* u1, cwo_c64* u2, double z);

/* Fresnel diffraction, Fourier form, Eq.(7)-(9): one transform instead of three,
 *   u2[m2,n2] = exp(i 2 pi z/lambda)/(i lambda z) px py exp(i pi (x2^2 + y2^2)/(lambda z))
 *               sum_{m1,n1} u1[m1,n1] exp(i pi (x1^2 + y1^2)/(lambda z)) exp(-i 2 pi (x1 x2 + y1 y2)/(lambda z)),
 * sample j of an axis at m = j - N/2 (Eq.(4)), x1 = m1 px, x2 = m2 p2x on the DESTINATION PITCH
 * p2x = lambda |z| / (Nx px), p2y = lambda |z| / (Ny py) (P:L158 is garbled; this is the pitch at which the kernel is the
 * DFT kernel).  z < 0: the kernel's sign flips (unnormalised inverse DFT).  z == 0 -> CWO_EINVAL. */
int cwo_fresnel_fourier(cwo_plan_t plan, const cwo_c64* u1, cwo_c64* u2, double z);

/* Shifted Fresnel diffraction, Eq.(10)-(14): Eq.(1) between a source plane of pitch (px, py) and a
 * destination plane of pitch (p1x, p1y) (cwo_plan_set_dst_pitch_xy) whose window is displaced by (ox, oy) metres
 * (cwo_plan_set_offset):
 *   u2[m1,n1] = exp(i 2 pi z/lambda)/(i lambda z) px py sum_{m0,n0} u1[m0,n0] exp(i pi ((x1-x0)^2 + (y1-y0)^2)/(lambda z)),
 *   x0 = m0 px, x1 = m1 p1x + ox (m = j - N/2), evaluated as the scaled convolution of Eq.(10) with the chirps of
 * Eq.(11)-(13).  With the default destination pitch and offset it equals cwo_fresnel_conv.  z == 0 -> CWO_EINVAL. */
int cwo_fresnel_shifted(cwo_plan_t plan, const cwo_c64* u1, cwo_c64* u2, double z);

/* 3-D diffraction as a stack of 2-D diffractions (Diffract3D): out[k] = cwo_asm(u1, zs[k]),
 * k = 0..n-1, the forward FFT of u1 computed once.  zs: HOST array of n doubles.  out: device,
 * [n][Ny][Nx] complex (float intensities with CWO_OPT_STACK_INTENSITY); must not overlap u1. */
int cwo_propagate_stack(cwo_plan_t plan, const cwo_c64* u1, const double* zs, int n, void* out);

/* Gerchberg-Saxton loop (section 7.2, Listing 8) between a source (hologram)
 * plane with amplitude amp_src and a destination (image) plane with amplitude amp_dst, z apart:
 *   G = amp_dst * exp(i phase_out);  p = phasor(P(-z)[G]);
 *   repeat iters times:  q = phasor(P(+z)[amp_src * p]);  p = phasor(P(-z)[amp_dst * q]);
 *   phase_out = atan2(Im p, Re p)  in [-pi, pi];   phasor(u) = u/|u|, 1 where u == 0.
 * P = cwo_fresnel_conv or cwo_asm per CWO_OPT_GS_METHOD.  phase_out is in/out (the library has no
 * random generator; the paper's SetRandPhase seed is unspecified).  iters == 0 yields the
 * kinoform of section 7.1.  amp_src, amp_dst, phase_out: float [Ny][Nx], device. */
int cwo_gs(cwo_plan_t plan, const float* amp_src, const float* amp_dst, double z, int iters,
           float* phase_out);

/* "Scale", Eq.(21): out[i] = (in[i] - min in)/(max in - min in) * 255 over n floats (an intensity field
 * of any shape, e.g. a whole stack); a constant field maps to 0.  in, out: device, 16-byte aligned; out == in allowed. */
int cwo_scale255(cwo_plan_t plan, const float* in, float* out, size_t n);

/* Scale (Eq.(21)) without a plan and without any allocation: the same map as cwo_scale255, bit for bit,
 * for callers that are not allowed to allocate device memory -- and therefore cannot call cwo_plan(), whose tables
 * (the {min, max} cell of Scale among them) come from cudaMalloc.  Typical cases: a thread working while a CUDA graph
 * is being captured elsewhere in the process in global mode (cudaMalloc is refused then), a component of a server or
 * plug-in host that owns all device memory through its own pool, a real-time loop that cannot afford the device-wide
 * synchronisation of cudaMalloc / cudaFree.
 *   in, out      DEVICE pointers to n floats, 16-byte aligned, owned by the caller; out == in allowed.
 *   cuda_stream  a cudaStream_t passed as void* (NULL: the null stream) on the CURRENT device; the call only enqueues
 *                three kernels on it and returns.
 *   cuda_error_out  may be NULL; receives the cudaError_t when the call returns CWO_ECUDA, else 0.
 * Scratch: per-chunk minima / maxima go to a fixed array compiled into libcwo.so (256.25 KiB of device memory on every
 * GPU that loads the library, held until the process exits), which bounds the size:
 *   n <= CWO_SCALE255_STATIC_MAX_N (2^28 floats = 1 GiB, a 16384 x 16384 plane); larger n returns CWO_ELIMIT and
 *   enqueues nothing.  n == 0, NULL or misaligned pointers: CWO_EINVAL.  Device not 10.x: CWO_EUNSUPPORTED.
 * The call itself never calls cudaMalloc, cudaFree or any allocating routine.  The FIRST call on each device looks up
 * the device address of the array (cudaGetSymbolAddress, once per device, with that device current); make that first
 * call outside any stream capture.
 * Every call on a GPU uses the same array, which keeps whatever the previous call left in it.  A call writes each
 * word before it reads it, so leftovers are harmless and nothing needs clearing -- but two calls that may run on the
 * GPU at the same time (streams with no ordering between them, or concurrent host threads) race on the array: keep
 * calls on one device ordered (one stream, or events). */
#define CWO_SCALE255_STATIC_MAX_N ((size_t)1 << 28)
int cwo_scale255_static(const float* in, float* out, size_t n, void* cuda_stream, int* cuda_error_out);

/* Computer-generated hologram of n point light sources, Eq.(23):
 *   out[j][i] = sum_k A_k cos( (2 pi/lambda) ((x - x_k)^2 + (y - y_k)^2)/(2 z_k) ),  (x, y) = ((i - Nx/2) px, (j - Ny/2) py),
 * on the plan's Nx x Ny grid, pitch and wavelength.  pts: DEVICE array of n x 4 doubles (x_k, y_k, z_k, A_k) [m, m, m, -];
 * z_k != 0.  out: float [Ny][Nx].  Direct O(n Nx Ny) sum (the paper's cwoPLS), no workspace. */
int cwo_pls_cgh(cwo_plan_t plan, const double* pts, int n, float* out);

const char* cwo_strerror(int code);
int cwo_last_cuda_error(cwo_plan_t plan);

#ifdef __cplusplus
}
#endif
#endif /* CWO_H_ */
