// scale_static.cu -- cwo_scale255_static (include/cwo.h): "Scale", Eq.(21), for callers that must not
// allocate device memory.
//
// Who needs it.  cwo_scale255 takes a plan, and cwo_plan() builds its tables with cudaMalloc -- the {min, max} cell that
// Scale reduces into is one of them.  Some callers cannot go through that: code that runs while another thread of the
// process is capturing a CUDA graph (cudaMalloc is refused for the whole process during a global-mode capture), code
// inside a server or plug-in host that has handed all of HBM to its own pool and forbids raw allocations, and
// real-time loops that cannot take the device-wide synchronisation a cudaMalloc / cudaFree implies.  For them the
// scratch of this variant lives in the library image itself: the file-scope array below, SS_SCRATCH_WORDS * 4 bytes
// (256.25 KiB), which every GPU that loads libcwo.so holds until the process exits.
//
// What differs from cwo_scale255.  The plan path reduces with atomicMin / atomicMax into a cell that two memsets
// re-arm before every call.  Here the field is cut into chunks of SS_CHUNK floats; a first kernel writes each chunk's
// {min, max} to its own slot of the array, a second one folds the slots into the {min, max} cell at the head of the
// array, and the map itself is the plan path's scale_kernel (outputs.cu) reading that cell.  Every word a call reads it
// has written itself earlier in the same call, so nothing has to start at zero and the previous call's leftovers are
// never looked at.  min and max do not depend on the order of reduction: the output is bit-identical to cwo_scale255's.
//
// The chunk slots bound the size: n <= CWO_SCALE255_STATIC_MAX_N = SS_MAX_CHUNKS * SS_CHUNK = 2^28 floats (1 GiB, one
// 16384 x 16384 intensity plane -- the largest plane the propagation calls accept).  Larger n -> CWO_ELIMIT.
//
// All calls on one GPU share the one array: two calls that can overlap on the GPU (different streams without an
// ordering between them, or two host threads) race on it.  Calls on one stream, or ordered by events, are safe.
#include <mutex>
#include <stdint.h>

#include "../../include/cwo.h"
#include "cwo_internal.h"

namespace {

constexpr int SS_THREADS = 256;
constexpr int SS_VEC = 8;                                              // float4 loads per thread and chunk
constexpr size_t SS_CHUNK = (size_t)SS_THREADS * 4 * SS_VEC;          // 8192 floats (32 KiB) per CTA
constexpr size_t SS_MAX_CHUNKS = CWO_SCALE255_STATIC_MAX_N / SS_CHUNK; // 32768
constexpr size_t SS_HEAD = 64;                                         // words: the {min, max} cell, padded to 256 bytes
constexpr size_t SS_SCRATCH_WORDS = SS_HEAD + 2 * SS_MAX_CHUNKS;
static_assert(CWO_SCALE255_STATIC_MAX_N % SS_CHUNK == 0, "the size limit is a whole number of chunks");

// [0] min, [1] max of the field (order-preserving integers, as outputs.cu); [SS_HEAD + 2c], [SS_HEAD + 2c + 1]: chunk c.
// In HOST code this name is only a handle for cudaGetSymbolAddress -- it is not a device address.
static __device__ __align__(256) unsigned g_scale_scratch[SS_SCRATCH_WORDS];

// the same order-preserving map float -> uint32 as outputs.cu (scale_kernel decodes the cell with its inverse)
__device__ __forceinline__ unsigned enc_f32(float f) {
    const unsigned u = __float_as_uint(f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

// {min, max} of a CTA's values -> out[0], out[1] (thread 0 writes)
template <int WARPS>
__device__ __forceinline__ void cta_minmax_store(unsigned lo, unsigned hi, unsigned* out) {
    __shared__ unsigned slo[WARPS], shi[WARPS];
    lo = __reduce_min_sync(0xffffffffu, lo);
    hi = __reduce_max_sync(0xffffffffu, hi);
    if ((threadIdx.x & 31) == 0) { slo[threadIdx.x >> 5] = lo; shi[threadIdx.x >> 5] = hi; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < WARPS; ++w) { lo = min(lo, slo[w]); hi = max(hi, shi[w]); }
        out[0] = lo; out[1] = hi;
    }
}

// CTA c reduces floats [c * SS_CHUNK, min(n, (c + 1) * SS_CHUNK)) -- never empty -- into part[2c], part[2c + 1]
__global__ void __launch_bounds__(SS_THREADS) chunk_minmax_kernel(const float* __restrict__ in, size_t n,
                                                                  unsigned* __restrict__ part) {
    const size_t base = (size_t)blockIdx.x * SS_CHUNK;
    const size_t end = base + SS_CHUNK < n ? base + SS_CHUNK : n;
    const size_t nvec = (end - base) / 4;
    const float4* in4 = reinterpret_cast<const float4*>(in + base);      // in is 16-byte aligned, base a multiple of 4
    unsigned lo = 0xffffffffu, hi = 0u;
    for (size_t i = threadIdx.x; i < nvec; i += SS_THREADS) {
        const float4 v = __ldcs(&in4[i]);
        const unsigned a = enc_f32(v.x), b = enc_f32(v.y), c = enc_f32(v.z), d = enc_f32(v.w);
        lo = min(min(lo, a), min(b, min(c, d)));
        hi = max(max(hi, a), max(b, max(c, d)));
    }
    for (size_t i = base + 4 * nvec + threadIdx.x; i < end; i += SS_THREADS) {
        const unsigned a = enc_f32(in[i]);
        lo = min(lo, a); hi = max(hi, a);
    }
    cta_minmax_store<SS_THREADS / 32>(lo, hi, part + 2 * (size_t)blockIdx.x);
}

// one CTA: fold the n_chunks slots into the cell mm[0..1]
__global__ void __launch_bounds__(1024) fold_minmax_kernel(const unsigned* __restrict__ part, unsigned n_chunks,
                                                           unsigned* __restrict__ mm) {
    unsigned lo = 0xffffffffu, hi = 0u;
    for (unsigned c = threadIdx.x; c < n_chunks; c += 1024) {
        const uint2 v = *reinterpret_cast<const uint2*>(part + 2 * (size_t)c);
        lo = min(lo, v.x); hi = max(hi, v.y);
    }
    cta_minmax_store<32>(lo, hi, mm);
}

// ---- set-up, once per device ---------------------------------------------------------------------------------------
struct StaticDevice { unsigned* scratch; int n_sm; bool ready; };
StaticDevice g_static_dev[cwo::MAX_DEVICES];
std::mutex g_static_mu;

// The current device's copy of g_scale_scratch.  cudaGetSymbolAddress resolves the symbol for the device that is current
// when it is called (each device has its own copy of the array), so the address is cached per device index.
int static_device(StaticDevice** out, int* cuda_error) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { *cuda_error = (int)e; return CWO_ECUDA; }
    if (dev < 0 || dev >= cwo::MAX_DEVICES) return CWO_EINVAL;
    std::lock_guard<std::mutex> lock(g_static_mu);
    StaticDevice& d = g_static_dev[dev];
    if (!d.ready) {
        int major = 0, n_sm = 0;
        if ((e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev)) != cudaSuccess ||
            (e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) {
            *cuda_error = (int)e;
            return CWO_ECUDA;
        }
        if (major != 10) return CWO_EUNSUPPORTED;
        void* ptr = nullptr;
        e = cudaGetSymbolAddress(&ptr, g_scale_scratch);
        if (e != cudaSuccess || !ptr) {
            *cuda_error = (int)e;
            return CWO_ECUDA;
        }
        d.scratch = static_cast<unsigned*>(ptr);
        d.n_sm = n_sm;
        d.ready = true;
    }
    *out = &d;
    return CWO_OK;
}

}  // namespace

extern "C" int cwo_scale255_static(const float* in, float* out, size_t n, void* cuda_stream, int* cuda_error_out) {
    int cuda_error = 0;
    if (cuda_error_out) *cuda_error_out = 0;
    if (!in || !out || ((uintptr_t)in & 15) || ((uintptr_t)out & 15) || n == 0) return CWO_EINVAL;
    if (n > CWO_SCALE255_STATIC_MAX_N) return CWO_ELIMIT;
    StaticDevice* d = nullptr;
    int rc = static_device(&d, &cuda_error);
    if (rc != CWO_OK) {
        if (cuda_error_out) *cuda_error_out = cuda_error;
        return rc;
    }
    cudaStream_t s = (cudaStream_t)cuda_stream;
    unsigned* mm = d->scratch;                      // device address of g_scale_scratch, not the host-side name
    unsigned* part = d->scratch + SS_HEAD;
    const unsigned n_chunks = (unsigned)((n + SS_CHUNK - 1) / SS_CHUNK);
    cudaError_t e;
    chunk_minmax_kernel<<<n_chunks, SS_THREADS, 0, s>>>(in, n, part);
    if ((e = cudaGetLastError()) == cudaSuccess) {
        fold_minmax_kernel<<<1, 1024, 0, s>>>(part, n_chunks, mm);
        if ((e = cudaGetLastError()) == cudaSuccess) e = cwo::launch_scale(in, out, n, mm, d->n_sm, s);
    }
    if (e != cudaSuccess) {
        if (cuda_error_out) *cuda_error_out = (int)e;
        return CWO_ECUDA;
    }
    return CWO_OK;
}
