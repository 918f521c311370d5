// dm_peaks.cu -- dm_measure_peaks (include/dm.h): the denominators DESIGN.md quotes for the rooflines of the
// psi update, measured on the device the library runs on (SURVEY.md 8(d) asks for the FP32 one explicitly):
// FP32 FMA issue rate (scalar and packed f32x2), HBM read-only and copy bandwidth, L2-resident read bandwidth,
// shared-memory read bandwidth.  Plain streaming kernels timed with CUDA events; no DM arithmetic here.
#include <cstdint>
#include <cstring>

#include <cuda_runtime.h>

#include "../../include/dm.h"

namespace {

constexpr int PK_NT = 256;

// 8 independent dependent-chains of FMAs per thread: ITER x 8 scalar FFMA
__global__ void __launch_bounds__(PK_NT) peak_ffma_kernel(float *out, int iters, float a, float b)
{
    float x[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) x[i] = (float)(threadIdx.x + i);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) x[i] = fmaf(x[i], a, b);
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += x[i];
    if (s == 123.456f) out[blockIdx.x * PK_NT + threadIdx.x] = s;
}

// the same with the packed two-lane instruction (FFMA2): ITER x 8 fma.rn.f32x2 = 16 lane-FMAs
__global__ void __launch_bounds__(PK_NT) peak_ffma2_kernel(float *out, int iters, float a, float b)
{
    unsigned long long x[8], aa, bb;
    asm volatile("mov.b64 %0, {%1, %1};\n" : "=l"(aa) : "f"(a));
    asm volatile("mov.b64 %0, {%1, %1};\n" : "=l"(bb) : "f"(b));
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const float v = (float)(threadIdx.x + i);
        asm volatile("mov.b64 %0, {%1, %1};\n" : "=l"(x[i]) : "f"(v));
    }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;\n" : "+l"(x[i]) : "l"(aa), "l"(bb));
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        float lo, hi;
        asm volatile("mov.b64 {%0, %1}, %2;\n" : "=f"(lo), "=f"(hi) : "l"(x[i]));
        s += lo + hi;
    }
    if (s == 123.456f) out[blockIdx.x * PK_NT + threadIdx.x] = s;
}

// grid-stride 128-bit reads of n float4, repeated `reps` times (reps > 1 on a small n = L2-resident)
__global__ void __launch_bounds__(PK_NT) peak_read_kernel(const float4 *src, size_t n, int reps, float *out)
{
    float s = 0.f;
    const size_t stride = (size_t)gridDim.x * PK_NT;
    for (int r = 0; r < reps; ++r) {
        size_t i = (size_t)blockIdx.x * PK_NT + threadIdx.x;
        for (; i + 3 * stride < n; i += 4 * stride) {
            const float4 v0 = __ldcg(src + i), v1 = __ldcg(src + i + stride), v2 = __ldcg(src + i + 2 * stride), v3 = __ldcg(src + i + 3 * stride);
            s += v0.x + v1.y + v2.z + v3.w;
        }
        for (; i < n; i += stride) s += __ldcg(src + i).x;
    }
    if (s == 123.456f) out[0] = s;
}

__global__ void __launch_bounds__(PK_NT) peak_copy_kernel(const float4 *src, float4 *dst, size_t n)
{
    const size_t stride = (size_t)gridDim.x * PK_NT;
    size_t i = (size_t)blockIdx.x * PK_NT + threadIdx.x;
    for (; i + 3 * stride < n; i += 4 * stride) {
        const float4 v0 = __ldcs(src + i), v1 = __ldcs(src + i + stride), v2 = __ldcs(src + i + 2 * stride), v3 = __ldcs(src + i + 3 * stride);
        __stcs(dst + i, v0); __stcs(dst + i + stride, v1); __stcs(dst + i + 2 * stride, v2); __stcs(dst + i + 3 * stride, v3);
    }
    for (; i < n; i += stride) __stcs(dst + i, __ldcs(src + i));
}

// conflict-free 128-bit shared-memory reads: 32 KiB per CTA, `iters` sweeps
__global__ void __launch_bounds__(PK_NT) peak_smem_kernel(float *out, int iters)
{
    __shared__ float4 buf[2048];
    for (int i = threadIdx.x; i < 2048; i += PK_NT) buf[i] = make_float4((float)i, 1.f, 2.f, 3.f);
    __syncthreads();
    float s0 = 0.f, s1 = 0.f, s2 = 0.f, s3 = 0.f;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int j = 0; j < 8; j += 4) {
            const float4 v0 = buf[(threadIdx.x + j * PK_NT + it) & 2047], v1 = buf[(threadIdx.x + (j + 1) * PK_NT + it) & 2047];
            const float4 v2 = buf[(threadIdx.x + (j + 2) * PK_NT + it) & 2047], v3 = buf[(threadIdx.x + (j + 3) * PK_NT + it) & 2047];
            s0 += v0.x; s1 += v1.y; s2 += v2.z; s3 += v3.w;
        }
    }
    const float s = s0 + s1 + s2 + s3;
    if (s == 123.456f) out[blockIdx.x] = s;
}

template <typename F> cudaError_t time_ms(cudaStream_t st, int warm, int reps, float *ms, F launch)
{
    cudaEvent_t e0, e1;
    cudaError_t e = cudaEventCreate(&e0);
    if (e != cudaSuccess) return e;
    e = cudaEventCreate(&e1);
    if (e != cudaSuccess) { cudaEventDestroy(e0); return e; }
    for (int i = 0; i < warm; ++i) launch();
    float best = 1e30f;
    for (int r = 0; r < reps && e == cudaSuccess; ++r) {
        cudaEventRecord(e0, st);
        launch();
        cudaEventRecord(e1, st);
        e = cudaEventSynchronize(e1);
        float t = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&t, e0, e1);
        if (t < best) best = t;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    *ms = best;
    return e != cudaSuccess ? e : cudaGetLastError();
}

} // namespace

extern "C" dm_status dm_measure_peaks(void *scratch_dev, size_t scratch_bytes, double *out_host, int n_out, void *stream)
{
    if (!scratch_dev || !out_host || n_out < 1) return DM_ERR_INVALID_ARG;
    if (scratch_bytes < ((size_t)512 << 20)) return DM_ERR_WORKSPACE;     // the streams must be much larger than L2
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return DM_ERR_CUDA;
    double r[DM_PEAK_FIELDS];
    memset(r, 0, sizeof r);
    float ms = 0.f;
    float *outf = (float *)scratch_dev;
    const int grid = sms * 8, iters = 1 << 14;
    // [0], [1]: FP32 lanes per second (one FMA = one lane-op), scalar and packed
    if (time_ms(st, 2, 5, &ms, [&] { peak_ffma_kernel<<<grid, PK_NT, 0, st>>>(outf, iters, 1.0001f, 0.5f); }) != cudaSuccess) return DM_ERR_CUDA;
    r[0] = (double)grid * PK_NT * iters * 8.0 / (ms * 1e-3);
    if (time_ms(st, 2, 5, &ms, [&] { peak_ffma2_kernel<<<grid, PK_NT, 0, st>>>(outf, iters, 1.0001f, 0.5f); }) != cudaSuccess) return DM_ERR_CUDA;
    r[1] = (double)grid * PK_NT * iters * 16.0 / (ms * 1e-3);
    // [2]: HBM read-only, [3]: HBM copy (read + write bytes), over the whole scratch
    const size_t n4 = scratch_bytes / sizeof(float4);
    if (time_ms(st, 1, 5, &ms, [&] { peak_read_kernel<<<grid, PK_NT, 0, st>>>((const float4 *)scratch_dev, n4, 1, outf); }) != cudaSuccess) return DM_ERR_CUDA;
    r[2] = (double)n4 * 16.0 / (ms * 1e-3) / 1e9;
    if (time_ms(st, 1, 5, &ms, [&] { peak_copy_kernel<<<grid, PK_NT, 0, st>>>((const float4 *)scratch_dev, (float4 *)scratch_dev + n4 / 2, n4 / 2); }) != cudaSuccess) return DM_ERR_CUDA;
    r[3] = (double)(n4 / 2) * 32.0 / (ms * 1e-3) / 1e9;
    // [4]: L2-resident reads: 32 MiB swept 64 times
    const size_t n_l2 = ((size_t)32 << 20) / sizeof(float4);
    if (time_ms(st, 1, 5, &ms, [&] { peak_read_kernel<<<grid, PK_NT, 0, st>>>((const float4 *)scratch_dev, n_l2, 64, outf); }) != cudaSuccess) return DM_ERR_CUDA;
    r[4] = (double)n_l2 * 16.0 * 64.0 / (ms * 1e-3) / 1e9;
    // [5]: shared-memory reads
    const int s_iters = 1 << 12;
    if (time_ms(st, 1, 5, &ms, [&] { peak_smem_kernel<<<grid, PK_NT, 0, st>>>(outf, s_iters); }) != cudaSuccess) return DM_ERR_CUDA;
    r[5] = (double)grid * PK_NT * s_iters * 8.0 * 16.0 / (ms * 1e-3) / 1e9;
    r[6] = (double)sms;
    for (int i = 0; i < n_out && i < DM_PEAK_FIELDS; ++i) out_host[i] = r[i];
    return DM_OK;
}
