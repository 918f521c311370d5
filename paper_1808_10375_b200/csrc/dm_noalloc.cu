// dm_noalloc.cu -- dm_probe_update_noalloc: the probe update of eq. (5) for callers who
// have no device workspace to lend and are not allowed to create one.
//
// Who that is.  The rest of this library keeps its intermediate sums in a workspace the caller allocates
// (dm_plan_set_workspace).  Some callers cannot do that: a plug-in inside a host application that handed
// every byte of device memory to its own pool at start-up, or an acquisition-time feedback loop in which
// cudaMalloc / cudaFree are banned because they synchronise the whole device (every stream stalls) and
// can fail once the pool owns the card.  Such a caller can still pass the arrays it already holds (its
// inputs and the output), but has nowhere to put the per-chunk partial sums of the two-stage reduction.
//
// What this file does about it.  The partial sums live in ONE file-scope __device__ array of
// DM_NOALLOC_SCRATCH_BYTES (16 MiB), which the CUDA driver places in device memory when this module is
// loaded on a GPU and keeps until the process exits: 16 MiB per GPU that uses the library, whether
// or not this entry point is ever called again.  The entry point itself calls no cudaMalloc, cudaFree,
// cudaMallocAsync or any library routine that allocates; problems whose partial sums do not fit are
// refused with DM_ERR_WORKSPACE and a text that names both sizes.
//
// The array's name is only meaningful to device code.  In host code it is a host-side shadow symbol, not
// a device address (a kernel handed `g_scratch` from the host would fault, or on a system where the
// GPU can reach host memory quietly use the wrong bytes), so the host side asks for the real address
// once per device with cudaGetSymbolAddress, with that device current, and passes the pointer it got to
// the kernels.  That set-up happens inside the first call on each device; make that first call outside
// any stream capture.
//
// Sharing.  Every call on a device uses the same array, and the array keeps whatever the previous call
// left in it.  Nothing in it has to start at zero: stage 1 writes every slot stage 2 reads (all pixels
// of all chunks of THIS call's geometry) before stage 2 reads it, on the same stream.  Two calls that
// overlap on the GPU (different streams, or different host threads on one device) race on the array and
// give wrong probes: order them yourself (one stream, or an event between them).
#include <cstdarg>
#include <cstdio>
#include <mutex>

#include "../../include/dm.h"

static __device__ __align__(256) unsigned char g_scratch[DM_NOALLOC_SCRATCH_BYTES];

namespace {

constexpr int NA_NT = 256;          // threads per CTA of both stages
constexpr int NA_MAX_DEVICES = 64;

struct DeviceSetup {
    bool done;
    unsigned char *scratch;         // device address of g_scratch on this device
    int sms;
};
DeviceSetup g_setup[NA_MAX_DEVICES];
std::mutex g_setup_mutex;

__device__ __forceinline__ float abs2(float2 a) { return a.x * a.x + a.y * a.y; }

// Stage 1.  CTA (bx, c): 2 * NA_NT probe pixels (thread t owns the pair r, r + 1), views j0 .. j1 of
// chunk c summed in ascending j, l ascending inside, for all K modes:
//   num_k(r) += conj(O_l(r + r_j)) * psi_jkl(r),   den(r) += |O_l(r + r_j)|^2      (eq. (5))
// written to pnum[c][k][r], pden[c][r] inside the static scratch.
template <int KT>
__global__ void __launch_bounds__(NA_NT) noalloc_probe_partial_kernel(
    int N, int L, int n_views, int chunk_len, int W, size_t HW, const int2 *__restrict__ pos,
    const float2 *__restrict__ O, const float2 *__restrict__ psi, float2 *__restrict__ pnum, float *__restrict__ pden)
{
    const int NN = N * N;
    const int r = 2 * (blockIdx.x * NA_NT + threadIdx.x);
    if (r >= NN) return;
    const int ry = r / N, rx = r % N;
    const int c = blockIdx.y, j0 = c * chunk_len, j1 = min(n_views, j0 + chunk_len);
    float4 num[KT];
#pragma unroll
    for (int k = 0; k < KT; ++k) num[k] = make_float4(0.f, 0.f, 0.f, 0.f);
    float den0 = 0.f, den1 = 0.f;
    for (int j = j0; j < j1; ++j) {
        const int2 p0 = __ldg(pos + j);                                   // (y0, x0)
        const float2 *ob = O + (size_t)(p0.x + ry) * W + p0.y + rx;
        const float2 *ps = psi + (size_t)j * KT * L * NN + r;
        for (int l = 0; l < L; ++l) {
            const float2 o0 = __ldg(ob + l * HW), o1 = __ldg(ob + l * HW + 1);
            den0 += abs2(o0);
            den1 += abs2(o1);
#pragma unroll
            for (int k = 0; k < KT; ++k) {
                const float4 s = __ldg(reinterpret_cast<const float4 *>(ps + (size_t)(k * L + l) * NN));
                num[k].x += o0.x * s.x + o0.y * s.y;
                num[k].y += o0.x * s.y - o0.y * s.x;
                num[k].z += o1.x * s.z + o1.y * s.w;
                num[k].w += o1.x * s.w - o1.y * s.z;
            }
        }
    }
#pragma unroll
    for (int k = 0; k < KT; ++k) *reinterpret_cast<float4 *>(pnum + ((size_t)c * KT + k) * NN + r) = num[k];
    *reinterpret_cast<float2 *>(pden + (size_t)c * NN + r) = make_float2(den0, den1);
}

// Stage 2.  Chunk-ascending FP64 sum of the partials, then the inertial quotient
//   P_new = (alpha P_old + num) / (alpha + den),   P_new = P_old where alpha + den = 0.
__global__ void __launch_bounds__(NA_NT) noalloc_probe_finalize_kernel(
    int NN, int K, int C, const float2 *__restrict__ pnum, const float *__restrict__ pden,
    const float2 *__restrict__ P_old, float2 *__restrict__ P_new, float alpha)
{
    const int r = blockIdx.x * NA_NT + threadIdx.x;
    const int k = blockIdx.y;
    if (r >= NN) return;
    double den = 0.0, nx = 0.0, ny = 0.0;
    for (int c = 0; c < C; ++c) {
        den += (double)pden[(size_t)c * NN + r];
        const float2 v = pnum[((size_t)c * K + k) * NN + r];
        nx += (double)v.x;
        ny += (double)v.y;
    }
    const float dd = alpha + (float)den;
    const float2 po = P_old[(size_t)k * NN + r];
    float2 pn = po;
    if (dd > 0.f) pn = make_float2((alpha * po.x + (float)nx) / dd, (alpha * po.y + (float)ny) / dd);
    P_new[(size_t)k * NN + r] = pn;
}

dm_status refuse(char *err, size_t cap, dm_status s, const char *fmt, ...)
{
    if (err && cap) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(err, cap, fmt, ap);
        va_end(ap);
    }
    return s;
}

} // namespace

extern "C" dm_status dm_probe_update_noalloc(int N, int n_views, int K, int L, int obj_h, int obj_w,
                                             const int32_t *positions_dev, const float *object_dev,
                                             const float *psi_dev, const float *probe_old_dev,
                                             float alpha_probe, float *probe_new_dev, void *stream,
                                             char *err_text_host, size_t err_text_bytes)
{
    char *const et = err_text_host;
    const size_t ec = err_text_bytes;
    if (et && ec) et[0] = 0;
    if (!positions_dev || !object_dev || !psi_dev || !probe_old_dev || !probe_new_dev)
        return refuse(et, ec, DM_ERR_INVALID_ARG, "dm_probe_update_noalloc: null pointer");
    if (n_views < 1 || K < 1 || L < 1 || obj_h < 1 || obj_w < 1 || !(alpha_probe >= 0.f))
        return refuse(et, ec, DM_ERR_INVALID_ARG, "dm_probe_update_noalloc: n_views, K, L, obj_h, obj_w must be >= 1 and alpha_probe >= 0");
    if (N != 64 && N != 128 && N != 256 && N != 512)
        return refuse(et, ec, DM_ERR_UNSUPPORTED, "dm_probe_update_noalloc: N = %d, must be 64, 128, 256 or 512", N);
    if (K * L > 8) return refuse(et, ec, DM_ERR_UNSUPPORTED, "dm_probe_update_noalloc: K * L = %d > 8", K * L);
    if (obj_h < N || obj_w < N)
        return refuse(et, ec, DM_ERR_OUT_OF_BOUNDS, "dm_probe_update_noalloc: object %d x %d smaller than the %d x %d window", obj_h, obj_w, N, N);

    // the size check comes before any CUDA call: one chunk of partial sums is the least that must fit
    const size_t NN = (size_t)N * N;
    const size_t per_chunk = NN * ((size_t)K * sizeof(float2) + sizeof(float));
    const size_t cap_chunks = (size_t)DM_NOALLOC_SCRATCH_BYTES / per_chunk;
    if (cap_chunks < 1)
        return refuse(et, ec, DM_ERR_WORKSPACE,
                      "dm_probe_update_noalloc: N = %d, K = %d needs %zu bytes of partial sums, the built-in scratch holds %zu "
                      "(use the plan API with a caller-allocated workspace)", N, K, per_chunk, (size_t)DM_NOALLOC_SCRATCH_BYTES);

    // once per device, with that device current: the device address of the static array + the SM count
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return refuse(et, ec, DM_ERR_CUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= NA_MAX_DEVICES) return refuse(et, ec, DM_ERR_UNSUPPORTED, "dm_probe_update_noalloc: device ordinal %d >= %d", dev, NA_MAX_DEVICES);
    DeviceSetup su;
    {
        std::lock_guard<std::mutex> lock(g_setup_mutex);
        if (!g_setup[dev].done) {
            void *ptr = nullptr;
            e = cudaGetSymbolAddress(&ptr, g_scratch);
            if (e != cudaSuccess || !ptr)
                return refuse(et, ec, DM_ERR_CUDA, "cudaGetSymbolAddress(scratch) on device %d: %s", dev, cudaGetErrorString(e));
            int sms = 0;
            e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
            if (e != cudaSuccess || sms < 1)
                return refuse(et, ec, DM_ERR_CUDA, "cudaDeviceGetAttribute(SM count) on device %d: %s", dev, cudaGetErrorString(e));
            g_setup[dev].scratch = static_cast<unsigned char *>(ptr);
            g_setup[dev].sms = sms;
            g_setup[dev].done = true;
        }
        su = g_setup[dev];
    }

    // geometry: as many view chunks as keep ~16 CTAs per SM in flight, but no more than fit the array
    const int blocks = (int)((NN / 2 + NA_NT - 1) / NA_NT);
    size_t chunks = ((size_t)su.sms * 16 + blocks - 1) / blocks;
    if (chunks > (size_t)n_views) chunks = (size_t)n_views;
    if (chunks > cap_chunks) chunks = cap_chunks;
    const int chunk_len = (int)((n_views + chunks - 1) / chunks);
    const int C = (n_views + chunk_len - 1) / chunk_len;

    float2 *pnum = reinterpret_cast<float2 *>(su.scratch);                                   // [C][K][NN]
    float *pden = reinterpret_cast<float *>(su.scratch + (size_t)C * K * NN * sizeof(float2)); // [C][NN]
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int2 *pos = reinterpret_cast<const int2 *>(positions_dev);
    const float2 *O = reinterpret_cast<const float2 *>(object_dev);
    const float2 *psi = reinterpret_cast<const float2 *>(psi_dev);
    const dim3 grid((unsigned)blocks, (unsigned)C);
#define NA_LAUNCH(KT)                                                                                        \
    noalloc_probe_partial_kernel<KT><<<grid, NA_NT, 0, st>>>(N, L, n_views, chunk_len, obj_w, (size_t)obj_h * obj_w, \
                                                             pos, O, psi, pnum, pden)
    switch (K) {
    case 1: NA_LAUNCH(1); break;
    case 2: NA_LAUNCH(2); break;
    case 3: NA_LAUNCH(3); break;
    case 4: NA_LAUNCH(4); break;
    case 5: NA_LAUNCH(5); break;
    case 6: NA_LAUNCH(6); break;
    case 7: NA_LAUNCH(7); break;
    default: NA_LAUNCH(8); break;
    }
#undef NA_LAUNCH
    noalloc_probe_finalize_kernel<<<dim3((unsigned)((NN + NA_NT - 1) / NA_NT), (unsigned)K), NA_NT, 0, st>>>(
        (int)NN, K, C, pnum, pden, reinterpret_cast<const float2 *>(probe_old_dev),
        reinterpret_cast<float2 *>(probe_new_dev), alpha_probe);
    e = cudaGetLastError();
    if (e != cudaSuccess) return refuse(et, ec, DM_ERR_CUDA, "dm_probe_update_noalloc launch: %s", cudaGetErrorString(e));
    return DM_OK;
}
