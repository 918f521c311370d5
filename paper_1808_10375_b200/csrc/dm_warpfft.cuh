// dm_warpfft.cuh -- warp-level register FFTs and the view-pipelined ("dataflow") psi update for
// every frame edge N in {64, 128, 256, 512} (steps S1-S6 of DESIGN.md; eqs. (2)-(4) of
// arXiv:1808.10375).  Included by dm_kernels.cuh.
//
// A frame of N >= 256 does not fit the registers / shared memory of one SM, so the 2-D FFT is
// split at the row / column boundary and the intermediate spectra travel through a small ring
// of scratch frames that stays resident in L2.  Every 1-D FFT is done by ONE WARP on 32 lanes x
// 32 registers with a single in-warp 32 x 32 transpose (no block barrier):
//
//   line of length N = 32 RX (RX = N/32 in {2,4,8,16});  a warp holds G = 32/RX lines;
//   register a = g RX + r of lane t holds element n = t + 32 r of line g
//   stage 1   radix-RX over r (-> k1), twiddle w_N^(t k1)
//   exchange  (lane t, reg a) -> (lane a, reg t)                        [xt_write / xt_read below]   
//   stage 2   radix-32 over t (-> k2):   frequency k = k1 + RX k2, held by lane a = g RX + k1
//
// Three phases per view, all running in ONE persistent kernel that pulls tasks from a queue in
// an order in which every task only depends on tasks queued before it (so a resident CTA never
// waits for a CTA that is not running):
//   A (rows)    R = 2 P O - psi, forward FFT along x, spectrum rows -> scratch ("column-group"
//               layout: group cg holds G adjacent kx as [y][c], 8 KiB contiguous)
//   B (columns) for all M = K L modes of one column group: forward FFT along y, mode-summed
//               modulus constraint (eq. (4)), inverse FFT along y, back to scratch in place
//   C (rows)    inverse FFT along x, psi_new = psi_old + beta (G - P O)
// Phase B of view v is queued D views after phase A of v, phase C another D views later; the
// window of views in flight (psi + scratch) is a few tens of MB, so psi_old of phase C and both
// scratch passes hit L2 and psi crosses HBM once in and once out.
//
// The FFT code is __host__ __device__: tests run it on the CPU through dm_host_fft2_path(path 4).
#pragma once
#include <cuda_runtime.h>

#include "dm_fft.cuh"
#include "dm_regfft.cuh"

namespace dmwf {

using namespace dmfft;

constexpr int WF_MAXW = 8;                           // warps per CTA: M = K L (2 if M = 1)
constexpr int WF_ROW = 272, WF_XBUF = 32 * WF_ROW;   // exchange buffer of one warp: 32 rows of 32 c64 + 16 B pad

// ---- in-warp 32 x 32 transpose (lane t, reg a) -> (lane a, reg t), one round -------------
// Every lane writes its 32 registers down a column (64-bit stores: the 16 lanes of a half warp
// fill 128 contiguous bytes) and reads one padded row back (128-bit loads, row stride 272 B:
// the 8 lanes of a quarter warp hit 8 different 16-byte bank groups).  No lane-dependent
// register choice, so no divergence.  wbuf = this warp's WF_XBUF bytes.
DM_HD void xt_write(const float2 (&u)[32], int t, unsigned char *wbuf)
{
#pragma unroll
    for (int a = 0; a < 32; ++a) *reinterpret_cast<float2 *>(wbuf + a * WF_ROW + t * 8) = u[a];
}
DM_HD void xt_read(float2 (&u)[32], int t, const unsigned char *wbuf)
{
#pragma unroll
    for (int b = 0; b < 32; b += 2) {
        const float4 v = *reinterpret_cast<const float4 *>(wbuf + t * WF_ROW + b * 8);
        u[b] = make_float2(v.x, v.y);
        u[b + 1] = make_float2(v.z, v.w);
    }
}

// ---- 1-D FFT of G lines by one warp (emulated lane by lane on the host) -----------------
// tw[k1 * 32 + t] = exp(-2 pi i t k1 / N)
template <int RX> DM_HD void stage1_fwd(float2 (&u)[32], const float2 *tw, int t)
{
    constexpr int G = 32 / RX;
#pragma unroll
    for (int g = 0; g < G; ++g) {
        float2 v[RX];
#pragma unroll
        for (int r = 0; r < RX; ++r) v[r] = u[g * RX + r];
        Dft<RX, false>::run(v);
        u[g * RX] = v[0];
#pragma unroll
        for (int k1 = 1; k1 < RX; ++k1) u[g * RX + k1] = cmul(v[k1], tw[k1 * 32 + t]);
    }
}

template <int RX> DM_HD void stage1_inv(float2 (&u)[32], const float2 *tw, int t)
{
    constexpr int G = 32 / RX;
#pragma unroll
    for (int g = 0; g < G; ++g) {
        float2 v[RX];
        v[0] = u[g * RX];
#pragma unroll
        for (int k1 = 1; k1 < RX; ++k1) v[k1] = cmulc(u[g * RX + k1], tw[k1 * 32 + t]);
        Dft<RX, true>::run(v);
#pragma unroll
        for (int r = 0; r < RX; ++r) u[g * RX + r] = v[r];
    }
}

// ---- layouts ------------------------------------------------------------------------------
// scratch frame: element (y, kx) at ((kx / G) N + y) G + kx % G        (G = 1024 / N columns per group)
template <int N> DM_HD int scratch_index(int y, int kx)
{
    constexpr int G = 1024 / N;
    return ((kx / G) * N + y) * G + kx % G;
}
// sqrt(I) storage: register k2 of lane a in column group cg sits at [cg][k2 >> 2][a][k2 & 3]
DM_HD int spec_pos(int cg, int a, int k2) { return ((cg * 8 + (k2 >> 2)) * 32 + a) * 4 + (k2 & 3); }
// natural-order frequency ky * N + kx held there after phase B's forward FFT
template <int N> DM_HD int spec_freq(int cg, int a, int k2)
{
    constexpr int RX = N / 32, G = 32 / RX;
    return ((a % RX) + RX * k2) * N + cg * G + a / RX;
}

} // namespace dmwf

// =========================================================================================
// The kernel (device only)
// =========================================================================================
#ifdef __CUDACC__

namespace dmwf {

struct WfArgs {
    int n_views, K, L, H, W;
    const int2 *pos;            // (y0, x0) per view
    const float2 *P;            // [K][N][N]
    const float2 *O;            // [L][H][W]
    float2 *psi;                // [n_views][M][N][N], updated in place
    const float *amp;           // [n_views][N*N] sqrt(I) in the layout of spec_pos
    const float2 *tw;           // [RX][32]
    float2 *scratch;            // [S][M][N*N] ring of spectrum frames
    int S, D;                   // ring slots, phase lag in views
    int nA, nB, nC;             // tasks per view and phase
    int *queue;                 // task counter
    int *cntA, *cntB, *cntC;    // [n_views] finished tasks per view and phase
    float *partF;               // [n_views * nB][2]  (eF_num, eF_den)
    float *partS;               // [n_views * nC][2]  (epsi_num, epsi_den)
    float beta, eps;
};

__device__ __forceinline__ void spin_until(const int *cnt, int want)
{
    int v;
    for (;;) {
        asm volatile("ld.acquire.gpu.global.s32 %0, [%1];\n" : "=r"(v) : "l"(cnt) : "memory");
        if (v >= want) break;
        __nanosleep(100);
    }
}

// 256-bit (one full 32-byte sector per lane) L2-only load / store of four adjacent complex values
__device__ __forceinline__ void ldcg256(const float2 *p, float2 &a, float2 &b, float2 &c, float2 &d)
{
    unsigned r0, r1, r2, r3, r4, r5, r6, r7;
    asm volatile("ld.global.cg.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];\n"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3), "=r"(r4), "=r"(r5), "=r"(r6), "=r"(r7) : "l"(p) : "memory");
    a = make_float2(__uint_as_float(r0), __uint_as_float(r1));
    b = make_float2(__uint_as_float(r2), __uint_as_float(r3));
    c = make_float2(__uint_as_float(r4), __uint_as_float(r5));
    d = make_float2(__uint_as_float(r6), __uint_as_float(r7));
}
__device__ __forceinline__ void stcg256(float2 *p, float2 a, float2 b, float2 c, float2 d)
{
    asm volatile("st.global.cg.v8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};\n"
                 :: "l"(p), "r"(__float_as_uint(a.x)), "r"(__float_as_uint(a.y)), "r"(__float_as_uint(b.x)), "r"(__float_as_uint(b.y)),
                    "r"(__float_as_uint(c.x)), "r"(__float_as_uint(c.y)), "r"(__float_as_uint(d.x)), "r"(__float_as_uint(d.y)) : "memory");
}

__device__ __forceinline__ float abs2_rn(float2 f) { return __fmaf_rn(f.y, f.y, __fmul_rn(f.x, f.x)); }

// forward / inverse 1-D FFT of the warp's G lines (registers <-> registers)
template <int RX> __device__ __forceinline__ void warp_fft_fwd(float2 (&u)[32], const float2 *s_tw, int t, unsigned char *wbuf)
{
    stage1_fwd<RX>(u, s_tw, t);
    xt_write(u, t, wbuf);
    __syncwarp();
    xt_read(u, t, wbuf);
    __syncwarp();
    dmreg::dft32<false>(u);
}
template <int RX> __device__ __forceinline__ void warp_fft_inv(float2 (&u)[32], const float2 *s_tw, int t, unsigned char *wbuf)
{
    dmreg::dft32<true>(u);
    xt_write(u, t, wbuf);
    __syncwarp();
    xt_read(u, t, wbuf);
    __syncwarp();
    stage1_inv<RX>(u, s_tw, t);
}

// One CTA = NW = blockDim.x / 32 warps (a multiple of M).  A task is NW row groups of a view
// (phases A, C) or NW / M column groups x M modes (phase B).
template <int N>
__global__ void __launch_bounds__(32 * WF_MAXW, 2) wf_dataflow_kernel(const WfArgs a)
{
    constexpr int RX = N / 32, G = 32 / RX, NN = N * N, NG = N / G;     // NG: column groups = row groups per frame
    extern __shared__ __align__(16) unsigned char smem[];
    __shared__ int s_task[2], s_go[2];
    __shared__ float red2[2][2 * WF_MAXW];

    const int tid = threadIdx.x, w = tid >> 5, t = tid & 31, NW = blockDim.x >> 5;
    const int M = a.K * a.L;
    unsigned char *wbuf = smem + w * WF_XBUF;                 // exchange buffer; doubles as the |F|^2 buffer
    float2 *s_tw = reinterpret_cast<float2 *>(smem + NW * WF_XBUF);       // [RX][32]
    // sqrt(I) of the task's column groups, staged by cp.async while the forward FFT runs: [NW / M][8][32] float4
    float4 *s_amp = reinterpret_cast<float4 *>(smem + NW * WF_XBUF + RX * 32 * sizeof(float2));
    for (int i = tid; i < RX * 32; i += blockDim.x) s_tw[i] = a.tw[i];
    const int T = a.nA + a.nB + a.nC;
    const int total = (a.n_views + 2 * a.D) * T;
    const int GPT = NW / M;                                               // column groups per B task

    // task -> (phase, sub, view); view outside [0, n_views) = nothing to do
    auto decode = [&](int task, int &phase, int &sub, int &view) {
        const int step = task / T, rem = task - step * T;
        if (rem < a.nA) { phase = 0; sub = rem; view = step; }
        else if (rem < a.nA + a.nB) { phase = 1; sub = rem - a.nA; view = step - a.D; }
        else { phase = 2; sub = rem - a.nA - a.nB; view = step - 2 * a.D; }
    };
    // thread 0: claim the next task that has work and wait for what it depends on (always tasks
    // queued earlier, hence finished or running on a resident CTA)
    auto resolve = [&](int task) -> int {
        for (;;) {
            if (task >= total) return task;
            int phase, sub, view;
            decode(task, phase, sub, view);
            if (view >= 0 && view < a.n_views) {
                if (phase == 0) { if (view >= a.S) spin_until(a.cntC + view - a.S, a.nC); }
                else if (phase == 1) spin_until(a.cntA + view, a.nA);
                else spin_until(a.cntB + view, a.nB);
                return task;
            }
            task = atomicAdd(a.queue, 1);
        }
    };
    if (tid == 0) s_task[0] = resolve(atomicAdd(a.queue, 1));
    __syncthreads();

    for (int buf = 0;; buf ^= 1) {
        const int task = s_task[buf];
        if (task >= total) break;
        int nxt = 0;
        if (tid == 0) nxt = atomicAdd(a.queue, 1);            // in flight while this task runs
        int phase, sub, view;
        decode(task, phase, sub, view);
        float2 *slot = a.scratch + (size_t)(view % a.S) * M * NN;
        const int2 p0 = a.pos[view];
        float2 u[32];
        bool active;
        float e0 = 0.f, e1 = 0.f;
        float *red = red2[buf];
        // A / C geometry: row group rgi of the view -> frame m, rows y0 .. y0 + G - 1
        const int rgi = sub * NW + w;
        const int m_ac = rgi / NG, y0 = (rgi % NG) * G;
        // B geometry: warp -> (column group, mode)
        const int cg = sub * GPT + w / M, m_b = w % M;
        // scratch address of (row y0 + t / RX, kx = t % RX) -- register k2 adds scratch_index(0, RX k2)
        const int sidx = scratch_index<N>(y0 + t / RX, t % RX);
        if (phase == 0) {
            // ---- S1 + S2: R = 2 P O - psi, G rows of one mode frame ----
            active = rgi < M * NG;
            if (active) {
                const int k = m_ac / a.L, l = m_ac % a.L;
                const float2 *psi_f = a.psi + ((size_t)view * M + m_ac) * NN + (size_t)y0 * N + t;
                const float2 *Pk = a.P + (size_t)k * NN + (size_t)y0 * N + t;
                const float2 *Ow = a.O + (size_t)l * a.H * a.W + (size_t)(p0.x + y0) * a.W + p0.y + t;
#pragma unroll
                for (int i = 0; i < 32; ++i) u[i] = __ldcs(psi_f + (i / RX) * N + (i % RX) * 32);   // streamed once: keep L1 for P and O
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    float2 p[16], o[16];
#pragma unroll
                    for (int i = 0; i < 16; ++i) {
                        const int e = 16 * h + i;
                        p[i] = __ldg(Pk + (e / RX) * N + (e % RX) * 32);
                        o[i] = __ldg(Ow + (size_t)(e / RX) * a.W + (e % RX) * 32);
                    }
#pragma unroll
                    for (int i = 0; i < 16; ++i) {
                        const float2 po = cmul(p[i], o[i]);
                        u[16 * h + i] = make_float2(2.f * po.x - u[16 * h + i].x, 2.f * po.y - u[16 * h + i].y);
                    }
                }
            }
        } else if (phase == 1) {
            // ---- spectrum rows of one column group, one mode: lane t holds y = t + 32 s ----
            active = (w < GPT * M) && (cg < NG);
            if (active) {
                // sqrt(I) of this column group comes from HBM and is only needed after the forward FFT:
                // copy it asynchronously into shared memory now (no registers held), one warp per group
                if (m_b == 0) {
                    const float4 *ampv = reinterpret_cast<const float4 *>(a.amp + (size_t)view * NN) + (size_t)cg * 256 + t;
                    const unsigned dst = (unsigned)__cvta_generic_to_shared(s_amp + (size_t)(w / M) * 256 + t);
#pragma unroll
                    for (int j = 0; j < 8; ++j)
                        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" :: "r"(dst + j * 512), "l"(ampv + j * 32) : "memory");
                    asm volatile("cp.async.commit_group;\n" ::: "memory");
                }
                const float2 *src = slot + (size_t)m_b * NN + (size_t)cg * N * G + (size_t)t * G;
#pragma unroll
                for (int s = 0; s < RX; ++s) {
                    if (G >= 4) {
#pragma unroll
                        for (int c = 0; c + 3 < G; c += 4)
                            ldcg256(src + (size_t)s * 32 * G + c, u[c * RX + s], u[(c + 1) * RX + s], u[(c + 2) * RX + s], u[(c + 3) * RX + s]);
                    } else {
#pragma unroll
                        for (int c = 0; c < G; c += 2) {
                            const float4 v = __ldcg(reinterpret_cast<const float4 *>(src + (size_t)s * 32 * G + c));
                            u[c * RX + s] = make_float2(v.x, v.y);
                            u[(c + 1) * RX + s] = make_float2(v.z, v.w);
                        }
                    }
                }
            }
        } else {
            // ---- scaled spectrum rows back from scratch: lane a = (g, k1), register k2 ----
            active = rgi < M * NG;
            if (active) {
                // psi_old is needed after the inverse FFT and may have left L2 since phase A read it
                {
                    const char *rows = reinterpret_cast<const char *>(a.psi + ((size_t)view * M + m_ac) * NN + (size_t)y0 * N);
#pragma unroll
                    for (int i = 0; i < 2; ++i) asm volatile("prefetch.global.L2 [%0];\n" :: "l"(rows + (size_t)(t + 32 * i) * 128));
                }
                const float2 *src = slot + (size_t)m_ac * NN + sidx;
#pragma unroll
                for (int k2 = 0; k2 < 32; ++k2) u[k2] = __ldcg(src + scratch_index<N>(0, RX * k2));
            }
        }
        // ---- forward FFT (A: along x, B: along y) ----
        if (phase != 2 && active) warp_fft_fwd<RX>(u, s_tw, t, wbuf);
        // ---- S4: mode-summed modulus constraint (eq. (4)) ----
        if (phase == 1) {
            float4 *mine = reinterpret_cast<float4 *>(wbuf) + t;
            if (active) {
#pragma unroll
                for (int j = 0; j < 8; ++j)
                    mine[j * 32] = make_float4(abs2_rn(u[4 * j]), abs2_rn(u[4 * j + 1]), abs2_rn(u[4 * j + 2]), abs2_rn(u[4 * j + 3]));
            }
            if (active && m_b == 0) asm volatile("cp.async.wait_all;\n" ::: "memory");
            __syncthreads();
            // reduce-scatter: the M warps of a column group share the 8 register rows j; the warp that owns row j
            // sums |F|^2 of all modes for it, forms the scale amp / sqrt(S) and leaves it where sqrt(I) was
            if (active) {
                float4 *ampv = s_amp + (size_t)(w / M) * 256 + t;
                const unsigned char *peers = smem + (size_t)(w - m_b) * WF_XBUF;
                const float cfac = 1.f / (float)NN;
                for (int j = m_b; j < 8; j += M) {
                    const float4 am = ampv[j * 32];
                    float4 S = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
                    for (int mm = 0; mm < WF_MAXW; ++mm)
                        if (mm < M) {
                            const float4 v = reinterpret_cast<const float4 *>(peers + (size_t)mm * WF_XBUF)[j * 32 + t];
                            S.x += v.x; S.y += v.y; S.z += v.z; S.w += v.w;
                        }
                    const float Sv[4] = {S.x, S.y, S.z, S.w}, av[4] = {am.x, am.y, am.z, am.w};
                    float sc[4];
#pragma unroll
                    for (int c = 0; c < 4; ++c) {
                        const float rs = rsqrtf(Sv[c] + a.eps);
                        const float d = Sv[c] * rs - av[c];
                        e0 = fmaf(d, d, e0);
                        e1 = fmaf(av[c], av[c], e1);
                        sc[c] = av[c] * rs * cfac;
                    }
                    ampv[j * 32] = make_float4(sc[0], sc[1], sc[2], sc[3]);
                }
            }
            __syncthreads();            // scales complete; every warp has read the |F|^2 buffers (they serve as exchange buffers again)
            if (active) {
                const float4 *scv = s_amp + (size_t)(w / M) * 256 + t;
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const float4 sc = scv[j * 32];
                    u[4 * j].x *= sc.x; u[4 * j].y *= sc.x;
                    u[4 * j + 1].x *= sc.y; u[4 * j + 1].y *= sc.y;
                    u[4 * j + 2].x *= sc.z; u[4 * j + 2].y *= sc.z;
                    u[4 * j + 3].x *= sc.w; u[4 * j + 3].y *= sc.w;
                }
            }
        }
        // ---- inverse FFT (B: along y, C: along x) ----
        if (phase != 0 && active) warp_fft_inv<RX>(u, s_tw, t, wbuf);
        // ---- stores ----
        if (phase == 0) {
            if (active) {
                float2 *dst = slot + (size_t)m_ac * NN + sidx;
#pragma unroll
                for (int k2 = 0; k2 < 32; ++k2) __stcg(dst + scratch_index<N>(0, RX * k2), u[k2]);
            }
        } else if (phase == 1) {
            if (active) {
                float2 *dst = slot + (size_t)m_b * NN + (size_t)cg * N * G + (size_t)t * G;
#pragma unroll
                for (int s = 0; s < RX; ++s) {
                    if (G >= 4) {
#pragma unroll
                        for (int c = 0; c + 3 < G; c += 4)
                            stcg256(dst + (size_t)s * 32 * G + c, u[c * RX + s], u[(c + 1) * RX + s], u[(c + 2) * RX + s], u[(c + 3) * RX + s]);
                    } else {
#pragma unroll
                        for (int c = 0; c < G; c += 2)
                            __stcg(reinterpret_cast<float4 *>(dst + (size_t)s * 32 * G + c),
                                   make_float4(u[c * RX + s].x, u[c * RX + s].y, u[(c + 1) * RX + s].x, u[(c + 1) * RX + s].y));
                    }
                }
            }
        } else {
            // ---- S6: psi_new = psi_old + beta (G - P O) ----
            if (active) {
                const int k = m_ac / a.L, l = m_ac % a.L;
                float2 *psi_f = a.psi + ((size_t)view * M + m_ac) * NN + (size_t)y0 * N + t;
                const float2 *Pk = a.P + (size_t)k * NN + (size_t)y0 * N + t;
                const float2 *Ow = a.O + (size_t)l * a.H * a.W + (size_t)(p0.x + y0) * a.W + p0.y + t;
#pragma unroll
                for (int h = 0; h < 4; ++h) {
                    float2 p[8], o[8], old[8];
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        const int e = 8 * h + i;
                        old[i] = __ldcs(psi_f + (e / RX) * N + (e % RX) * 32);
                        p[i] = __ldg(Pk + (e / RX) * N + (e % RX) * 32);
                        o[i] = __ldg(Ow + (size_t)(e / RX) * a.W + (e % RX) * 32);
                    }
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        const int e = 8 * h + i;
                        const float2 po = cmul(p[i], o[i]);
                        const float tx = u[e].x - po.x, ty = u[e].y - po.y;
                        const float2 nw = make_float2(fmaf(a.beta, tx, old[i].x), fmaf(a.beta, ty, old[i].y));
                        e0 = fmaf(tx, tx, fmaf(ty, ty, e0));
                        e1 = fmaf(nw.x, nw.x, fmaf(nw.y, nw.y, e1));
                        __stcs(psi_f + (e / RX) * N + (e % RX) * 32, nw);
                    }
                }
            }
        }
        // ---- publish: partial sums (fixed order), completion counter, next task ----
        if (phase != 0) {
#pragma unroll
            for (int s = 16; s > 0; s >>= 1) {
                e0 += __shfl_xor_sync(0xffffffffu, e0, s);
                e1 += __shfl_xor_sync(0xffffffffu, e1, s);
            }
            if (t == 0) { red[w] = e0; red[WF_MAXW + w] = e1; }
        }
        // thread 0 looks at the next task's dependency counter NOW: the round trip of that acquire load
        // overlaps with the barrier and the release below instead of following them
        const int *dep = nullptr;
        int want = 0, seen = 0;
        bool early = false;
        if (tid == 0 && nxt < total) {
            int nphase, nsub, nview;
            decode(nxt, nphase, nsub, nview);
            if (nview >= 0 && nview < a.n_views) {
                early = true;
                if (nphase == 0) { if (nview >= a.S) { dep = a.cntC + nview - a.S; want = a.nC; } }
                else if (nphase == 1) { dep = a.cntA + nview; want = a.nA; }
                else { dep = a.cntB + nview; want = a.nB; }
                if (dep) asm volatile("ld.acquire.gpu.global.s32 %0, [%1];\n" : "=r"(seen) : "l"(dep) : "memory");
            }
        }
        // if the next task can start (the common case), publish it with the barrier that ends this one:
        // the other warps go on while thread 0 writes the partial sums and releases the completion count
        if (tid == 0) {
            // (pays with many warps per CTA; with 2 or 3 the warp of thread 0 would be the straggler of the next task)
            const bool go = NW >= 6 && early && (dep == nullptr || seen >= want);
            s_go[buf] = go;
            if (go) s_task[buf ^ 1] = nxt;
        }
        __syncthreads();
        const bool go = s_go[buf] != 0;
        if (tid == 0) {
            if (phase != 0) {
                float s0 = 0.f, s1 = 0.f;
                for (int ww = 0; ww < NW; ++ww) { s0 += red[ww]; s1 += red[WF_MAXW + ww]; }
                float2 *out = reinterpret_cast<float2 *>(phase == 1 ? a.partF : a.partS) +
                              ((size_t)view * (phase == 1 ? a.nB : a.nC) + sub);
                *out = make_float2(phase == 2 ? s0 * a.beta * a.beta : s0, s1);
            }
            __threadfence();
            atomicAdd((phase == 0 ? a.cntA : phase == 1 ? a.cntB : a.cntC) + view, 1);
            if (!go) {
                if (early) {
                    if (dep) spin_until(dep, want);
                    s_task[buf ^ 1] = nxt;
                } else {
                    s_task[buf ^ 1] = resolve(nxt);
                }
            }
        }
        if (!go) __syncthreads();
    }
}

} // namespace dmwf
#endif // __CUDACC__
