// dm_kernels.cuh -- sm_100a kernels of the multi-mode difference-map iteration
// (arXiv:1808.10375 Sec. II).  Included by dm_api.cu only.
//
//   psi update (S1-S6, eqs. (2)-(4)):
//     fused_frame_kernel<N>   N in {64,128}: one CTA per mode frame, frame resident in shared
//                             memory, the K*L CTAs of a view form a thread-block cluster and
//                             sum |F|^2 over modes through distributed shared memory.
//     rows_fwd / cols_mod / rows_inv   any N: the same passes split at the row/column
//                             boundary, intermediate spectra in an L2-sized scratch.
//   object update (S7, eq. (6)):  object_gather_kernel   (coverage lists, no atomics)
//   probe  update (S8, eq. (5)):  probe_partial_kernel + probe_finalize_kernel
//   errors (S9, eq. (7)):         error_finalize_kernel
#pragma once
#include <cooperative_groups.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "dm_fft.cuh"
#include "dm_regfft.cuh"
#include "dm_warpfft.cuh"

namespace cg = cooperative_groups;
using namespace dmfft;

// ------------------------------------------------------------------ helpers ---------
struct BlockSync { __device__ __forceinline__ void operator()() const { __syncthreads(); } };

// deterministic block sum of NV values per thread: xor-shuffle tree inside each warp, then
// thread 0 adds the warp sums in warp order.  red needs NV * 32 floats.  Result in thread 0.
template <int NV>
__device__ __forceinline__ void block_sum(float (&v)[NV], float *red)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
#pragma unroll
    for (int i = 0; i < NV; ++i) {
#pragma unroll
        for (int s = 16; s > 0; s >>= 1) v[i] += __shfl_xor_sync(0xffffffffu, v[i], s);
    }
    __syncthreads();
    if (lane == 0) {
#pragma unroll
        for (int i = 0; i < NV; ++i) red[i * 32 + warp] = v[i];
    }
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int i = 0; i < NV; ++i) {
            float s = 0.f;
            for (int w = 0; w < nw; ++w) s += red[i * 32 + w];
            v[i] = s;
        }
    }
}

__device__ __forceinline__ float4 ld4(const float2 *p) { return *reinterpret_cast<const float4 *>(p); }
__device__ __forceinline__ void st4(float2 *p, float4 v) { *reinterpret_cast<float4 *>(p) = v; }

// P*O for two adjacent pixels: p = (P[r], P[r+1]) as float4, o0/o1 the two object pixels
__device__ __forceinline__ float4 po2(float4 p, float2 o0, float2 o1)
{
    return make_float4(p.x * o0.x - p.y * o0.y, p.x * o0.y + p.y * o0.x,
                       p.z * o1.x - p.w * o1.y, p.z * o1.y + p.w * o1.x);
}

// ------------------------------------------------------------- set_data kernels -----
// amp[v][p] = sqrt(I[v][spec[p]]): sqrt(I) stored once in the spectrum layout of the chosen
// psi-update path (spec[p] = natural-order frequency index ky*N + kx held at storage position p)
__global__ void amp_permute_kernel(int N, const float *__restrict__ inten, const int *__restrict__ spec,
                                   float *__restrict__ amp, size_t total)
{
    const size_t NN = (size_t)N * N;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const size_t v = i / NN;
        amp[i] = sqrtf(inten[v * NN + spec[i % NN]]);
    }
}

// psi_jkl = P_k * O_l|window   (eq. (2))
__global__ void psi_init_kernel(int N, int K, int L, int H, int W, const int2 *__restrict__ pos,
                                const float2 *__restrict__ P, const float2 *__restrict__ O,
                                float2 *__restrict__ psi)
{
    const int NN = N * N, M = K * L;
    const int f = blockIdx.y;                 // mode frame index j*M + k*L + l
    const int j = f / M, m = f % M, k = m / L, l = m % L;
    const int2 p0 = pos[j];
    const float2 *Ow = O + (size_t)l * H * W + (size_t)p0.x * W + p0.y;
    const float2 *Pk = P + (size_t)k * NN;
    float2 *out = psi + (size_t)f * NN;
    for (int r = blockIdx.x * blockDim.x + threadIdx.x; r < NN; r += gridDim.x * blockDim.x) {
        const int ry = r / N, rx = r % N;
        out[r] = cmul(Pk[r], Ow[(size_t)ry * W + rx]);
    }
}

// single-CTA max of n floats, scaled: out[0] = factor * max(x)
__global__ void max_scale_kernel(const float *__restrict__ x, size_t n, float factor, float *out)
{
    __shared__ float red[32];
    float m = 0.f;
    for (size_t i = threadIdx.x; i < n; i += blockDim.x) m = fmaxf(m, x[i]);
    for (int s = 16; s > 0; s >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, s));
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < (int)(blockDim.x >> 5); ++w) m = fmaxf(m, red[w]);
        out[0] = factor * m;
    }
}

// ------------------------------------------------------------ fused psi update ------
struct PsiArgs {
    int n_views, K, L, H, W;
    const int2 *pos;            // (y0, x0) per view
    const float2 *P;            // [K][N][N]   current probe
    const float2 *O;            // [L][H][W]   current object
    float2 *psi;                // [n_views][K][L][N][N], updated in place
    const float *amp;           // [n_views][N][N] sqrt(I) in spectrum layout
    const float2 *tw;           // [N] exp(-2 pi i n/N)
    float beta, eps;
    float *part;                // fused: [n_views*M][4] ; staged: see dm_api.cu
    // staged path only
    float2 *scratch;            // [chunk][M][N][N]
    int view0, n_chunk;         // first view and number of views of this chunk
    float *part2;               // staged: second partial array
};

// One CTA = one mode frame of one view; cluster = the M = K*L frames of the view.
// Steps: S1 P*O, S2 R = 2PO - psi, S3 FFT2 (in shared memory), S4 mode-summed modulus
// (|F|^2 summed over the cluster through DSMEM), S5 IFFT2, S6 psi += beta (G - PO).
template <int N, int NT>
__global__ void __launch_bounds__(NT, 1) fused_frame_kernel(const PsiArgs a)
{
    constexpr int NN = N * N;
    cg::cluster_group cluster = cg::this_cluster();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *tile = reinterpret_cast<float2 *>(smem_raw);      // NN complex, swizzled
    float *sbuf = reinterpret_cast<float *>(tile + NN);         // NN floats: |F|^2 partial, then scale
    float2 *tw = reinterpret_cast<float2 *>(sbuf + NN);         // N twiddles
    __shared__ float red[4 * 32];

    const int tid = threadIdx.x;
    const int M = a.K * a.L;
    const int m = (int)cluster.block_rank();
    const int view = blockIdx.x / M;
    const int k = m / a.L, l = m % a.L;
    const int2 p0 = a.pos[view];
    const float2 *Pk = a.P + (size_t)k * NN;
    const float2 *Ow = a.O + (size_t)l * a.H * a.W + (size_t)p0.x * a.W + p0.y;
    float2 *psi = a.psi + ((size_t)view * M + m) * NN;
    const float *ampv = a.amp + (size_t)view * NN;

    for (int i = tid; i < N; i += NT) tw[i] = a.tw[i];

    // S1 + S2: R = 2 P O - psi, two pixels (16 B) per step
    for (int c = tid; c < NN / 2; c += NT) {
        const int e = 2 * c, ry = e / N, rx = e % N;
        const float4 ps = ld4(psi + e);
        const float4 pp = __ldg(reinterpret_cast<const float4 *>(Pk + e));
        const float2 *o = Ow + (size_t)ry * a.W + rx;
        const float4 po = po2(pp, __ldg(o), __ldg(o + 1));
        st4(tile + swz(e), make_float4(2.f * po.x - ps.x, 2.f * po.y - ps.y, 2.f * po.z - ps.z, 2.f * po.w - ps.w));
    }
    __syncthreads();
    // S3: forward 2-D FFT, rows then columns
    axis_fft<N, false, false, N, N>(tile, tw, tid, NT, BlockSync());
    axis_fft<N, false, true, N, N>(tile, tw, tid, NT, BlockSync());

    // S4: S(q) = sum over the cluster of |F_m(q)|^2
    for (int e = tid; e < NN; e += NT) sbuf[e] = cabs2(tile[swz(e)]);
    cluster.sync();
    float acc[4] = {0.f, 0.f, 0.f, 0.f};
    {
        const int lo = (int)(((long long)NN * m / M) & ~3LL), hi = (m == M - 1) ? NN : (int)(((long long)NN * (m + 1) / M) & ~3LL);
        const float inv_nn = 1.f / (float)NN;
        for (int e = lo + tid; e < hi; e += NT) {
            float S = 0.f;
            for (int mm = 0; mm < M; ++mm) S += cluster.map_shared_rank(sbuf, mm)[e];
            const float amp = ampv[e];
            const float d = sqrtf(S) - amp;
            acc[0] += d * d;
            acc[1] += amp * amp;
            sbuf[e] = amp / sqrtf(S + a.eps) * inv_nn;      // scale incl. the 1/N^2 of the inverse
        }
    }
    cluster.sync();
    for (int mm = 0; mm < M; ++mm) {
        const int lo = (int)(((long long)NN * mm / M) & ~3LL), hi = (mm == M - 1) ? NN : (int)(((long long)NN * (mm + 1) / M) & ~3LL);
        const float *g = cluster.map_shared_rank(sbuf, mm);
        for (int e = lo + tid; e < hi; e += NT) {
            const float s = g[e];
            float2 f = tile[swz(e)];
            tile[swz(e)] = make_float2(f.x * s, f.y * s);
        }
    }
    cluster.sync();     // peers have finished reading this CTA's sbuf; also a block barrier
    // S5: inverse 2-D FFT, columns then rows (mirror of the forward passes)
    axis_fft<N, true, true, N, N>(tile, tw, tid, NT, BlockSync());
    axis_fft<N, true, false, N, N>(tile, tw, tid, NT, BlockSync());

    // S6: psi_new = psi_old + beta (G - PO)
    for (int c = tid; c < NN / 2; c += NT) {
        const int e = 2 * c, ry = e / N, rx = e % N;
        const float4 ps = ld4(psi + e);
        const float4 pp = __ldg(reinterpret_cast<const float4 *>(Pk + e));
        const float2 *o = Ow + (size_t)ry * a.W + rx;
        const float4 po = po2(pp, __ldg(o), __ldg(o + 1));
        const float4 g = ld4(tile + swz(e));
        const float4 d = make_float4(a.beta * (g.x - po.x), a.beta * (g.y - po.y), a.beta * (g.z - po.z), a.beta * (g.w - po.w));
        const float4 nw = make_float4(ps.x + d.x, ps.y + d.y, ps.z + d.z, ps.w + d.w);
        acc[2] += d.x * d.x + d.y * d.y + d.z * d.z + d.w * d.w;
        acc[3] += nw.x * nw.x + nw.y * nw.y + nw.z * nw.z + nw.w * nw.w;
        st4(psi + e, nw);
    }
    block_sum<4>(acc, red);
    if (tid == 0) {
        float4 *out = reinterpret_cast<float4 *>(a.part) + blockIdx.x;
        *out = make_float4(acc[0], acc[1], acc[2], acc[3]);
    }
}

// ------------------------------------------------------------ staged psi update -----
// Tile of ROWS x N per CTA: R = 2PO - psi, forward row FFT, spectrum rows to scratch.
template <int N, int ROWS, int NT>
__global__ void __launch_bounds__(NT) rows_fwd_kernel(const PsiArgs a)
{
    constexpr int NN = N * N, TE = ROWS * N;
    __shared__ __align__(16) float2 tile[TE];
    __shared__ float2 tw[N];
    const int tid = threadIdx.x;
    const int M = a.K * a.L;
    constexpr int TPF = N / ROWS;                       // tiles per frame
    const int fl = blockIdx.x / TPF, row0 = (blockIdx.x % TPF) * ROWS;   // frame index inside the chunk
    const int view = a.view0 + fl / M, m = fl % M, k = m / a.L, l = m % a.L;
    const int2 p0 = a.pos[view];
    const float2 *Pk = a.P + (size_t)k * NN + (size_t)row0 * N;
    const float2 *Ow = a.O + (size_t)l * a.H * a.W + (size_t)(p0.x + row0) * a.W + p0.y;
    const float2 *psi = a.psi + ((size_t)view * M + m) * NN + (size_t)row0 * N;
    for (int i = tid; i < N; i += NT) tw[i] = a.tw[i];
    for (int c = tid; c < TE / 2; c += NT) {
        const int e = 2 * c, ry = e / N, rx = e % N;
        const float4 ps = ld4(psi + e);
        const float4 pp = __ldg(reinterpret_cast<const float4 *>(Pk + e));
        const float2 *o = Ow + (size_t)ry * a.W + rx;
        const float4 po = po2(pp, __ldg(o), __ldg(o + 1));
        st4(tile + swz(e), make_float4(2.f * po.x - ps.x, 2.f * po.y - ps.y, 2.f * po.z - ps.z, 2.f * po.w - ps.w));
    }
    __syncthreads();
    axis_fft<N, false, false, N, ROWS>(tile, tw, tid, NT, BlockSync());
    float2 *out = a.scratch + (size_t)fl * NN + (size_t)row0 * N;
    for (int c = tid; c < TE / 2; c += NT) st4(out + 2 * c, ld4(tile + swz(2 * c)));
}

// One CTA = (view, strip of SW spectrum columns), all M modes: forward column FFT, mode-summed
// modulus constraint (eq. (4)), inverse column FFT, back to scratch in place.
template <int N, int SW, int NT>
__global__ void __launch_bounds__(NT) cols_mod_kernel(const PsiArgs a)
{
    constexpr int NN = N * N, TE = N * SW;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *tiles = reinterpret_cast<float2 *>(smem_raw);       // [M][N][SW]
    __shared__ float2 tw[N];
    __shared__ float red[2 * 32];
    const int tid = threadIdx.x;
    const int M = a.K * a.L;
    const int strip = blockIdx.x, vl = blockIdx.y, view = a.view0 + vl;
    float2 *base = a.scratch + (size_t)vl * M * NN + strip * SW;
    for (int i = tid; i < N; i += NT) tw[i] = a.tw[i];
    for (int c = tid; c < M * TE / 2; c += NT) {
        const int mm = c / (TE / 2), e = 2 * (c % (TE / 2)), y = e / SW, xs = e % SW;
        st4(tiles + mm * TE + swz(e), ld4(base + (size_t)mm * NN + (size_t)y * N + xs));
    }
    __syncthreads();
    for (int mm = 0; mm < M; ++mm) axis_fft<N, false, true, SW, N>(tiles + mm * TE, tw, tid, NT, BlockSync());
    float acc[2] = {0.f, 0.f};
    const float *ampv = a.amp + (size_t)view * NN + strip * SW;
    const float inv_nn = 1.f / (float)NN;
    for (int e = tid; e < TE; e += NT) {
        const int se = swz(e);
        float S = 0.f;
        for (int mm = 0; mm < M; ++mm) S += cabs2(tiles[mm * TE + se]);
        const float amp = ampv[(size_t)(e / SW) * N + (e % SW)];
        const float d = sqrtf(S) - amp;
        acc[0] += d * d;
        acc[1] += amp * amp;
        const float s = amp / sqrtf(S + a.eps) * inv_nn;
        for (int mm = 0; mm < M; ++mm) {
            float2 f = tiles[mm * TE + se];
            tiles[mm * TE + se] = make_float2(f.x * s, f.y * s);
        }
    }
    __syncthreads();
    for (int mm = 0; mm < M; ++mm) axis_fft<N, true, true, SW, N>(tiles + mm * TE, tw, tid, NT, BlockSync());
    for (int c = tid; c < M * TE / 2; c += NT) {
        const int mm = c / (TE / 2), e = 2 * (c % (TE / 2)), y = e / SW, xs = e % SW;
        st4(base + (size_t)mm * NN + (size_t)y * N + xs, ld4(tiles + mm * TE + swz(e)));
    }
    block_sum<2>(acc, red);
    if (tid == 0) {
        float2 *out = reinterpret_cast<float2 *>(a.part) + ((size_t)view * (N / SW) + strip);
        *out = make_float2(acc[0], acc[1]);
    }
}

// Inverse row FFT of the scratch rows, then psi_new = psi_old + beta (G - PO).
template <int N, int ROWS, int NT>
__global__ void __launch_bounds__(NT) rows_inv_kernel(const PsiArgs a)
{
    constexpr int NN = N * N, TE = ROWS * N;
    __shared__ __align__(16) float2 tile[TE];
    __shared__ float2 tw[N];
    __shared__ float red[2 * 32];
    const int tid = threadIdx.x;
    const int M = a.K * a.L;
    constexpr int TPF = N / ROWS;
    const int fl = blockIdx.x / TPF, row0 = (blockIdx.x % TPF) * ROWS;
    const int view = a.view0 + fl / M, m = fl % M, k = m / a.L, l = m % a.L;
    const int2 p0 = a.pos[view];
    const float2 *Pk = a.P + (size_t)k * NN + (size_t)row0 * N;
    const float2 *Ow = a.O + (size_t)l * a.H * a.W + (size_t)(p0.x + row0) * a.W + p0.y;
    float2 *psi = a.psi + ((size_t)view * M + m) * NN + (size_t)row0 * N;
    const float2 *in = a.scratch + (size_t)fl * NN + (size_t)row0 * N;
    for (int i = tid; i < N; i += NT) tw[i] = a.tw[i];
    for (int c = tid; c < TE / 2; c += NT) st4(tile + swz(2 * c), ld4(in + 2 * c));
    __syncthreads();
    axis_fft<N, true, false, N, ROWS>(tile, tw, tid, NT, BlockSync());
    float acc[2] = {0.f, 0.f};
    for (int c = tid; c < TE / 2; c += NT) {
        const int e = 2 * c, ry = e / N, rx = e % N;
        const float4 ps = ld4(psi + e);
        const float4 pp = __ldg(reinterpret_cast<const float4 *>(Pk + e));
        const float2 *o = Ow + (size_t)ry * a.W + rx;
        const float4 po = po2(pp, __ldg(o), __ldg(o + 1));
        const float4 g = ld4(tile + swz(e));
        const float4 d = make_float4(a.beta * (g.x - po.x), a.beta * (g.y - po.y), a.beta * (g.z - po.z), a.beta * (g.w - po.w));
        const float4 nw = make_float4(ps.x + d.x, ps.y + d.y, ps.z + d.z, ps.w + d.w);
        acc[0] += d.x * d.x + d.y * d.y + d.z * d.z + d.w * d.w;
        acc[1] += nw.x * nw.x + nw.y * nw.y + nw.z * nw.z + nw.w * nw.w;
        st4(psi + e, nw);
    }
    block_sum<2>(acc, red);
    if (tid == 0) {
        float2 *out = reinterpret_cast<float2 *>(a.part2) + ((size_t)(view * M + m) * TPF + row0 / ROWS);
        *out = make_float2(acc[0], acc[1]);
    }
}

// --------------------------------------------------------------- object update ------
// eq. (6): one thread per object pixel, one CTA per TH x TW tile; the tile's
// covering views come from the precomputed coverage list (ascending j), k ascending inside:
// the same summation order as the definition, no atomics.  Uses the OLD probe and new psi.
//   O_new = (alpha O_old + num) / (alpha + den)   (alpha + den == 0: keep O_old)
constexpr int OBJ_TH = 8, OBJ_TW = 32, OBJ_NT = OBJ_TH * OBJ_TW, OBJ_LMAX = 8;

// KT = compile-time K (0: run-time K).  With KT > 0 the covering views are processed in batches
// of U = 8 / (KT LT) views whose psi and P loads are all issued before the first use (memory-level
// parallelism); a view that does not contain the pixel contributes exact zeros, so the sum and
// its order are those of the definition.
template <int KT, int LT>
__global__ void __launch_bounds__(OBJ_NT) object_gather_kernel(
    int N, int K_rt, int H, int W, const int2 *__restrict__ pos, const int *__restrict__ tile_ptr,
    const int *__restrict__ tile_views, const float2 *__restrict__ P, const float2 *__restrict__ psi,
    const float2 *__restrict__ O_old, float2 *__restrict__ O_new, const float *__restrict__ alphas,
    float *__restrict__ part /* [tiles][LT][2] */, float *__restrict__ den_out /* may be NULL */)
{
    __shared__ int s_j[OBJ_NT];
    __shared__ int2 s_p[OBJ_NT];
    __shared__ float red[2 * LT * 32];
    const int K = KT ? KT : K_rt;
    const int NN = N * N;
    const int ntx = (W + OBJ_TW - 1) / OBJ_TW;
    const int tile = blockIdx.x, ty = tile / ntx, tx = tile % ntx;
    const int y = ty * OBJ_TH + threadIdx.x / OBJ_TW, x = tx * OBJ_TW + threadIdx.x % OBJ_TW;
    const bool inb = (y < H) && (x < W);
    float2 num[LT];
    float den = 0.f;
#pragma unroll
    for (int l = 0; l < LT; ++l) num[l] = make_float2(0.f, 0.f);
    const int beg = tile_ptr[tile], end = tile_ptr[tile + 1];
    const size_t vstride = (size_t)K * LT * NN;
    for (int b0 = beg; b0 < end; b0 += OBJ_NT) {
        const int nb = min(OBJ_NT, end - b0);
        __syncthreads();
        if ((int)threadIdx.x < nb) {
            const int j = tile_views[b0 + threadIdx.x];
            s_j[threadIdx.x] = j;
            s_p[threadIdx.x] = pos[j];
        }
        __syncthreads();
        if (!inb) continue;
        int i = 0;
        if (KT > 0) {
            constexpr int KK = KT > 0 ? KT : 1;
            constexpr int U = (8 / (KK * LT)) > 0 ? (8 / (KK * LT)) : 1;
            for (; i + U <= nb; i += U) {
                float2 pv[U][KK], sv[U][KK][LT];
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    const int ry = y - s_p[i + u].x, rx = x - s_p[i + u].y;
                    const bool ok = (unsigned)ry < (unsigned)N && (unsigned)rx < (unsigned)N;
                    const int r = ok ? ry * N + rx : 0;
                    const float2 *ps = psi + (size_t)s_j[i + u] * vstride + r;
#pragma unroll
                    for (int k = 0; k < KK; ++k) {
                        pv[u][k] = ok ? __ldg(P + (size_t)k * NN + r) : make_float2(0.f, 0.f);
#pragma unroll
                        for (int l = 0; l < LT; ++l)
                            sv[u][k][l] = ok ? __ldg(ps + (size_t)(k * LT + l) * NN) : make_float2(0.f, 0.f);
                    }
                }
#pragma unroll
                for (int u = 0; u < U; ++u)
#pragma unroll
                    for (int k = 0; k < KK; ++k) {
                        const float2 p = pv[u][k];
                        den += cabs2(p);
#pragma unroll
                        for (int l = 0; l < LT; ++l) {
                            const float2 sx = sv[u][k][l];
                            num[l].x += p.x * sx.x + p.y * sx.y;
                            num[l].y += p.x * sx.y - p.y * sx.x;
                        }
                    }
            }
        }
        for (; i < nb; ++i) {
            const int ry = y - s_p[i].x, rx = x - s_p[i].y;
            if ((unsigned)ry < (unsigned)N && (unsigned)rx < (unsigned)N) {
                const int r = ry * N + rx;
                const float2 *ps = psi + (size_t)s_j[i] * vstride + r;
                for (int k = 0; k < K; ++k) {
                    const float2 p = __ldg(P + (size_t)k * NN + r);
                    den += cabs2(p);
#pragma unroll
                    for (int l = 0; l < LT; ++l) {
                        const float2 sx = __ldg(ps + (size_t)(k * LT + l) * NN);
                        num[l].x += p.x * sx.x + p.y * sx.y;
                        num[l].y += p.x * sx.y - p.y * sx.x;
                    }
                }
            }
        }
    }
    float acc[2 * LT];
#pragma unroll
    for (int i = 0; i < 2 * LT; ++i) acc[i] = 0.f;
    if (inb) {
        const float alpha = alphas[0];
        const float dd = alpha + den;
        if (den_out) den_out[(size_t)y * W + x] = den;
#pragma unroll
        for (int l = 0; l < LT; ++l) {
            const size_t o = (size_t)l * H * W + (size_t)y * W + x;
            const float2 oo = O_old[o];
            float2 on = oo;
            if (dd > 0.f) on = make_float2((alpha * oo.x + num[l].x) / dd, (alpha * oo.y + num[l].y) / dd);
            O_new[o] = on;
            acc[2 * l] = cabs2(csub(on, oo));
            acc[2 * l + 1] = cabs2(on);
        }
    }
    block_sum<2 * LT>(acc, red);
    if (threadIdx.x == 0) {
#pragma unroll
        for (int i = 0; i < 2 * LT; ++i) part[(size_t)tile * 2 * LT + i] = acc[i];
    }
}

// ---------------------------------------------------------------- probe update ------
// eq. (5), stage 1: each CTA sums a contiguous chunk of views (j ascending, l
// ascending inside) for 512 probe pixels and all K modes; uses the NEW object and new psi.
constexpr int PRB_NT = 256;

template <int KT>
__global__ void __launch_bounds__(PRB_NT) probe_partial_kernel(
    int N, int L, int n_views, int chunk_len, int H, int W, const int2 *__restrict__ pos,
    const float2 *__restrict__ O, const float2 *__restrict__ psi, float2 *__restrict__ pnum /* [C][K][NN] */,
    float *__restrict__ pden /* [C][NN] */)
{
    const int NN = N * N;
    const int r = 2 * (blockIdx.x * PRB_NT + threadIdx.x);
    if (r >= NN) return;
    const int ry = r / N, rx = r % N;
    const int c = blockIdx.y, j0 = c * chunk_len, j1 = min(n_views, j0 + chunk_len);
    float4 num[KT];
#pragma unroll
    for (int k = 0; k < KT; ++k) num[k] = make_float4(0.f, 0.f, 0.f, 0.f);
    float den0 = 0.f, den1 = 0.f;
    const size_t HW = (size_t)H * W;
    int j = j0;
    if (L == 1) {
        // L = 1 (every config but c3): UV views per step, all of their psi / O loads issued before the
        // first use (memory-level parallelism); the sums keep the order j ascending
        constexpr int UV = KT <= 2 ? 4 : 2;
        for (; j + UV <= j1; j += UV) {
            float4 sv[UV][KT];
            float2 o0[UV], o1[UV];
#pragma unroll
            for (int u = 0; u < UV; ++u) {
                const int2 p0 = __ldg(pos + j + u);
                const float2 *ob = O + (size_t)(p0.x + ry) * W + p0.y + rx;
                o0[u] = __ldg(ob);
                o1[u] = __ldg(ob + 1);
#pragma unroll
                for (int k = 0; k < KT; ++k)
                    sv[u][k] = __ldg(reinterpret_cast<const float4 *>(psi + ((size_t)(j + u) * KT + k) * NN + r));
            }
#pragma unroll
            for (int u = 0; u < UV; ++u) {
                den0 += cabs2(o0[u]);
                den1 += cabs2(o1[u]);
#pragma unroll
                for (int k = 0; k < KT; ++k) {
                    const float4 s = sv[u][k];
                    num[k].x += o0[u].x * s.x + o0[u].y * s.y;
                    num[k].y += o0[u].x * s.y - o0[u].y * s.x;
                    num[k].z += o1[u].x * s.z + o1[u].y * s.w;
                    num[k].w += o1[u].x * s.w - o1[u].y * s.z;
                }
            }
        }
    }
    for (; j < j1; ++j) {
        const int2 p0 = __ldg(pos + j);
        const float2 *ob = O + (size_t)(p0.x + ry) * W + p0.y + rx;
        const float2 *ps = psi + (size_t)j * KT * L * NN + r;
        for (int l = 0; l < L; ++l) {
            const float2 o0 = __ldg(ob + l * HW), o1 = __ldg(ob + l * HW + 1);
            den0 += cabs2(o0);
            den1 += cabs2(o1);
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

// stage 2: fixed-order (chunk ascending) FP64 sum of the partials, inertial quotient, eq. (7) partials.
// grid = (pixel blocks, K): one probe mode per blockIdx.y (the shared denominator is re-summed per mode).
__global__ void __launch_bounds__(256) probe_finalize_kernel(
    int N, int K, int C, const float2 *__restrict__ pnum, const float *__restrict__ pden,
    const float2 *__restrict__ P_old, float2 *__restrict__ P_new, const float *__restrict__ alphas,
    float *__restrict__ part /* [blocks][K][2] */, float *__restrict__ den_out /* may be NULL */)
{
    __shared__ float red[2 * 32];
    const int NN = N * N;
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    const int k = blockIdx.y;
    const bool inb = r < NN;
    float acc[2] = {0.f, 0.f};
    if (inb) {
        double den = 0.0, nx = 0.0, ny = 0.0;
        int c = 0;
        for (; c + 8 <= C; c += 8) {
            float d[8];
            float2 v[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                d[u] = pden[(size_t)(c + u) * NN + r];
                v[u] = pnum[((size_t)(c + u) * K + k) * NN + r];
            }
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                den += (double)d[u];
                nx += (double)v[u].x;
                ny += (double)v[u].y;
            }
        }
        for (; c < C; ++c) {
            den += (double)pden[(size_t)c * NN + r];
            const float2 v = pnum[((size_t)c * K + k) * NN + r];
            nx += (double)v.x;
            ny += (double)v.y;
        }
        const float alpha = alphas[1];
        const float denf = (float)den, dd = alpha + denf;
        if (den_out && k == 0) den_out[r] = denf;
        const float2 po = P_old[(size_t)k * NN + r];
        float2 pn = po;
        if (dd > 0.f) pn = make_float2((alpha * po.x + (float)nx) / dd, (alpha * po.y + (float)ny) / dd);
        P_new[(size_t)k * NN + r] = pn;
        acc[0] = cabs2(csub(pn, po));
        acc[1] = cabs2(pn);
    }
    block_sum<2>(acc, red);
    if (threadIdx.x == 0) {
        part[((size_t)blockIdx.x * K + k) * 2] = acc[0];
        part[((size_t)blockIdx.x * K + k) * 2 + 1] = acc[1];
    }
}

// -------------------------------------------------------------- mode diagnostics ----
// out[m] = sum over the n elements of mode m of |x|^2 (FP64, fixed order).
__global__ void __launch_bounds__(1024) mode_power_kernel(const float2 *__restrict__ x, size_t n, double *__restrict__ out)
{
    __shared__ double sh[1024];
    const float2 *p = x + (size_t)blockIdx.x * n;
    double acc = 0.0;
    for (size_t i = threadIdx.x; i < n; i += 1024) acc += (double)p[i].x * (double)p[i].x + (double)p[i].y * (double)p[i].y;
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int w = 512; w > 0; w >>= 1) {
        if ((int)threadIdx.x < w) sh[threadIdx.x] += sh[threadIdx.x + w];
        __syncthreads();
    }
    if (threadIdx.x == 0) out[blockIdx.x] = sh[0];
}

// ---------------------------------------------------------------------- errors ------
// One CTA per column of the error row: fixed-order FP64 sums of (num, den) partial pairs,
// value = sqrt(num/den), 0/0 := 0   (eq. (7); A10).
struct ErrArgs {
    const float *pF;  int nF, sF;        // pairs at pF[i*sF], pF[i*sF+1]
    const float *pS;  int nS, sS;        // psi pairs
    const float *pP;  int nP;            // [nP][K][2]
    const float *pO;  int nO;            // [nO][L][2]
    int K, L;
    double *row;
};

constexpr int ERR_NT = 1024;

__global__ void __launch_bounds__(ERR_NT) error_finalize_kernel(const ErrArgs a)
{
    __shared__ double sn[ERR_NT], sd[ERR_NT];
    const int q = blockIdx.x;
    const float *p; int n, s;
    if (q == 0)            { p = a.pF; n = a.nF; s = a.sF; }
    else if (q == 1)       { p = a.pS; n = a.nS; s = a.sS; }
    else if (q < 2 + a.K)  { p = a.pP + 2 * (q - 2); n = a.nP; s = 2 * a.K; }
    else                   { p = a.pO + 2 * (q - 2 - a.K); n = a.nO; s = 2 * a.L; }
    // fixed order: thread t sums i = t, t + NT, ... (four loads in flight), then a binary tree over t
    double num = 0.0, den = 0.0;
    int i = threadIdx.x;
    for (; i + 3 * ERR_NT < n; i += 4 * ERR_NT) {
        float vn[4], vd[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            vn[u] = p[(size_t)(i + u * ERR_NT) * s];
            vd[u] = p[(size_t)(i + u * ERR_NT) * s + 1];
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            num += (double)vn[u];
            den += (double)vd[u];
        }
    }
    for (; i < n; i += ERR_NT) {
        num += (double)p[(size_t)i * s];
        den += (double)p[(size_t)i * s + 1];
    }
    sn[threadIdx.x] = num;
    sd[threadIdx.x] = den;
    __syncthreads();
    for (int w = ERR_NT / 2; w > 0; w >>= 1) {
        if ((int)threadIdx.x < w) {
            sn[threadIdx.x] += sn[threadIdx.x + w];
            sd[threadIdx.x] += sd[threadIdx.x + w];
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) a.row[q] = sd[0] > 0.0 ? sqrt(sn[0] / sd[0]) : 0.0;
}
