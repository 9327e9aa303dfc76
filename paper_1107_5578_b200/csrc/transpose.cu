// transpose.cu -- out[c][r] = in[r][c] for complex64 and float32 fields, through 32 x 32 shared-memory tiles.
// The separable Fresnel path (lineconv_kernel.cuh) convolves whole contiguous lines; between its row pass and its
// column pass the field is turned once, so both read and write full 256-byte segments (8 N^2 bytes in, 8 N^2 out).
#include "cwo_internal.h"

namespace cwo {

template <typename T>
__global__ void __launch_bounds__(256) transpose_kernel(const T* __restrict__ in, T* __restrict__ out, int rows, int cols) {
    __shared__ T tile[32][33];
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const int c0 = blockIdx.x * 32, r0 = blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < 4; ++k) tile[ty + 8 * k][tx] = in[(size_t)(r0 + ty + 8 * k) * cols + c0 + tx];
    __syncthreads();
#pragma unroll
    for (int k = 0; k < 4; ++k) out[(size_t)(c0 + ty + 8 * k) * rows + r0 + tx] = tile[tx][ty + 8 * k];
}

// out[c][r] = real field of in[r][c] -- |u|^2 (Eq.(20)), |u|, Re u, Im u or the phase (Eq.(25)): the last
// transposition of the separable Fresnel forms when the call returns a real field -- 8 N^2 bytes in, 4 N^2 out, no
// separate conversion pass
__global__ void __launch_bounds__(256) transpose_real_kernel(const float2* __restrict__ in, float* __restrict__ out, int rows,
                                                             int cols, int mode) {
    __shared__ float tile[32][33];
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const int c0 = blockIdx.x * 32, r0 = blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const float2 v = in[(size_t)(r0 + ty + 8 * k) * cols + c0 + tx];
        tile[ty + 8 * k][tx] = real_field(v.x, -v.y, 1.0f, mode);
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < 4; ++k) out[(size_t)(c0 + ty + 8 * k) * rows + r0 + tx] = tile[tx][ty + 8 * k];
}

template <typename T>
static cudaError_t launch_transpose(const T* in, T* out, int rows, int cols, cudaStream_t s) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(cols / 32), (unsigned)(rows / 32)); cfg.blockDim = dim3(256);
    cfg.dynamicSmemBytes = 0; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, transpose_kernel<T>, in, out, rows, cols);
}

cudaError_t launch_transpose_c64(const float2* in, float2* out, int rows, int cols, cudaStream_t s) {
    return launch_transpose<float2>(in, out, rows, cols, s);
}
cudaError_t launch_transpose_f32(const float* in, float* out, int rows, int cols, cudaStream_t s) {
    return launch_transpose<float>(in, out, rows, cols, s);
}
cudaError_t launch_transpose_real(const float2* in, float* out, int rows, int cols, int real_mode, cudaStream_t s) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(cols / 32), (unsigned)(rows / 32)); cfg.blockDim = dim3(256);
    cfg.dynamicSmemBytes = 0; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, transpose_real_kernel, in, out, rows, cols, real_mode);
}

}  // namespace cwo
