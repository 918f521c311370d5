// dm_vtfft.cuh -- path 6: TWO whole 128 x 128 frames in flight per SM.  Steps S1-S6 of DESIGN.md; eqs. (2)-(4) of
// arXiv:1808.10375.
//
// Path 3 (dm_regfft.cuh) gives one frame all 64 K registers of an SM, so the memory-side phases of a frame and its
// FFT passes run one after another.  Path 5 (dm_pairfft.cuh) put two HALF frames on an SM, but each half pays the
// whole latency chain of a frame (barriers, L2 round trips, DSMEM exchange), so nothing was won.  Here every CTA of
// 256 threads owns a WHOLE frame and two CTAs share an SM: each thread plays two of path 3's 512 "virtual threads"
// (virtual warp vw = 8 v + w, v = 0, 1) one after the other, with the same register layouts, passes, twiddles and
// spectrum layout.  The virtual thread that is not running is parked in tensor memory (64 words per virtual thread,
// 128 of the CTA's 256 columns x 128 lanes = its whole half of the SM's TMEM).  What changes against path 3:
//   * exchange 2 runs out of tensor memory: per round z every virtual thread moves 16 registers TMEM -> shared
//     (64 KiB buffer, the layout of dmreg::x2_write) and 16 back; exchange 1 is warp-local as before
//   * no tensor memory is left for psi_old and P*O: S6 reads psi_old, P and O a second time.  psi is prefetched into
//     L2 one frame ahead and its S1 loads carry an evict-last hint, its S6 loads evict-first, so the second read is
//     an L2 hit and psi still crosses HBM once in, once out
//   * the M = K*L frames of a view sit on M consecutive CTAs and meet at a release / acquire counter in L2
// One latency chain now covers a whole frame, and the other CTA of the SM fills its gaps.
#pragma once
#include "dm_regfft.cuh"

#ifdef __CUDACC__
namespace dmvt {

using namespace dmreg;

constexpr int VNT = 256;
constexpr int V_XBUF = 65536;                    // exchange 2, one round; exchange 1 (8 warps x 4608 B) aliases it
constexpr int VT_SMEM = V_XBUF + 2048;
constexpr int SPIN_LIMIT = 1 << 22;

#ifdef DM_VT_PROF
#define VPROF(i) { const long long now_ = clock64(); prof[i] += now_ - tprev; tprev = now_; }
#else
#define VPROF(i)
#endif

struct VtArgs {
    int n_views, K, L, H, W;
    const int2 *pos;
    const float2 *P, *O;
    float2 *psi;
    const float *amp;
    const float2 *wy, *wx;
    float4 *sbuf;               // [2][frames in flight][8][512]
    float *part;                // [grid][4]
    float beta, eps;
    int *gbar;                  // [groups]
};

__device__ __forceinline__ uint64_t l2_policy(bool last)
{
    uint64_t p;
    if (last) asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;\n" : "=l"(p));
    else asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;\n" : "=l"(p));
    return p;
}
__device__ __forceinline__ float2 ld_l2hint(const float2 *p, uint64_t policy)
{
    float2 v;
    asm volatile("ld.global.L1::no_allocate.L2::cache_hint.v2.f32 {%0, %1}, [%2], %3;\n" : "=f"(v.x), "=f"(v.y) : "l"(p), "l"(policy) : "memory");
    return v;
}

// park / fetch NE complex registers u[E0 .. E0 + NE) at words 2 E0 .. of the virtual thread's 64-word TMEM slot
template <int E0, int NE> __device__ __forceinline__ void park(const float2 (&u)[32], uint32_t slot)
{
#pragma unroll
    for (int e = E0; e < E0 + NE; e += 4) tmem_st8(slot + 2 * e, u[e], u[e + 1], u[e + 2], u[e + 3]);
}
template <int E0, int NE> __device__ __forceinline__ void fetch(float2 (&u)[32], uint32_t slot)
{
#pragma unroll
    for (int e = E0; e < E0 + NE; e += 4) tmem_ld8(slot + 2 * e, u[e], u[e + 1], u[e + 2], u[e + 3]);
}

// exchange 2, round z, for both virtual threads: 16 registers each TMEM -> shared, barrier, shared -> TMEM
__device__ __forceinline__ void x2_round(int z, int w, int t, uint32_t slot0, uint32_t slot1, float2 *xb)
{
    float2 h[2][16];
#pragma unroll
    for (int v = 0; v < 2; ++v) {
        const uint32_t s = (v ? slot1 : slot0) + 32u * z;
#pragma unroll
        for (int i = 0; i < 16; i += 4) tmem_ld8(s + 2 * i, h[v][i], h[v][i + 1], h[v][i + 2], h[v][i + 3]);
    }
    tmem_wait_ld();
#pragma unroll
    for (int v = 0; v < 2; ++v) {
        float2 *p = xb + (8 * v + w) * 32 + t;
#pragma unroll
        for (int c = 0; c < 16; ++c) p[c * 512] = h[v][c];
    }
    __syncthreads();
#pragma unroll
    for (int v = 0; v < 2; ++v) {
        const float2 *p = xb + (8 * v + w) * 512 + t;
#pragma unroll
        for (int i = 0; i < 16; ++i) h[v][i] = p[i * 32];
    }
#pragma unroll
    for (int v = 0; v < 2; ++v) {
        const uint32_t s = (v ? slot1 : slot0) + 32u * z;
#pragma unroll
        for (int i = 0; i < 16; i += 4) tmem_st8(s + 2 * i, h[v][i], h[v][i + 1], h[v][i + 2], h[v][i + 3]);
    }
    tmem_wait_st();
    __syncthreads();
}

// grid = frames in flight (2 per SM); frame slot f = blockIdx.x holds mode f % M of view group f / M
template <int MT>
__global__ void __launch_bounds__(VNT, 2) vtfft128_kernel(const VtArgs a)
{
    extern __shared__ __align__(128) unsigned char smem[];
    unsigned char *xbuf = smem;
    float2 *xb2 = reinterpret_cast<float2 *>(xbuf);
    float2 *s_wy = reinterpret_cast<float2 *>(smem + V_XBUF);
    float2 *s_wx = s_wy + 128;
    __shared__ float red[4 * 8];
    __shared__ uint32_t s_tmem;

    const int tid = threadIdx.x, w = tid >> 5, t = tid & 31;
    const int M = MT ? MT : a.K * a.L;
    const int slot = blockIdx.x, nslots = gridDim.x;
    const int m = slot % M, cl = slot / M, ncl = nslots / M;
    const int k = m / a.L, l = m % a.L;
    if (tid < 128) s_wy[tid] = a.wy[tid];
    else s_wx[tid - 128] = a.wx[tid - 128];
    if (w == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n"
                     :: "r"((uint32_t)__cvta_generic_to_shared(&s_tmem)), "r"(256) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
    // this thread's 128 private words: lane quarter w % 4, column block (w / 4) * 128; two 64-word slots
    const uint32_t slot0 = s_tmem + ((uint32_t)(32 * (w & 3)) << 16) + (uint32_t)(w >> 2) * 128u;
    const uint32_t slot1 = slot0 + 64u;

    unsigned char *wbuf = xbuf + w * X1_WARP;
    const uint64_t keep = l2_policy(true), drop = l2_policy(false);
    const float cfac = a.beta > 0.f ? 1.f / (float)RNN : 0.f;
    float e0 = 0.f, e1 = 0.f, e2 = 0.f, e3 = 0.f;
    int par = 0, it = 0;
    bool alive = true;

#ifdef DM_VT_PROF
    long long prof[8] = {0, 0, 0, 0, 0, 0, 0, 0}, tprev = clock64();
#endif
    for (int view = cl; cl < ncl && view < a.n_views; view += ncl, par ^= 1, ++it) {
        const int2 p0 = a.pos[view];
        float2 *frame = a.psi + ((size_t)view * M + m) * RNN;
        const float2 *Ofr = a.O + (size_t)l * a.H * a.W + (size_t)p0.x * a.W + p0.y;
        const float2 *Pfr = a.P + (size_t)k * RNN;
        // the next frame of this CTA: into L2 now (128 KiB = 4 lines of 128 B per thread), read by S1 one frame later
        if (view + ncl < a.n_views) {
            const char *nx = reinterpret_cast<const char *>(a.psi + ((size_t)(view + ncl) * M + m) * RNN) + (size_t)tid * 128;
#pragma unroll
            for (int i = 0; i < 4; ++i) asm volatile("prefetch.global.L2::evict_last [%0];\n" :: "l"(nx + (size_t)i * 32768));
        }
        // ---- S1-S3 (first half): R = 2 P O - psi, pass 1, exchange 1, pass 2; parked ----
#pragma unroll 1
        for (int v = 0; v < 2; ++v) {
            const int vw = 8 * v + w;
            const float2 *Pk = Pfr + vw * RN + t, *Ow = Ofr + (size_t)vw * a.W + t, *ps = frame + vw * RN + t;
            float2 u[32];
#pragma unroll
            for (int e = 0; e < 32; ++e) u[e] = __ldg(Pk + (e >> 2) * 16 * RN + (e & 3) * 32);
#pragma unroll
            for (int h = 0; h < 4; ++h) {
                float2 q[8], o[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const int ee = 8 * h + e;
                    o[e] = __ldg(Ow + (size_t)(ee >> 2) * 16 * a.W + (ee & 3) * 32);
                    q[e] = ld_l2hint(ps + (ee >> 2) * 16 * RN + (ee & 3) * 32, keep);
                }
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const int ee = 8 * h + e;
                    const float2 po = cmul(u[ee], o[e]);
                    u[ee] = make_float2(2.f * po.x - q[e].x, 2.f * po.y - q[e].y);
                }
            }
            {
                float2 wy[8], wx[4];
#pragma unroll
                for (int q = 0; q < 8; ++q) wy[q] = s_wy[vw * 8 + q];
#pragma unroll
                for (int r = 0; r < 4; ++r) wx[r] = s_wx[t * 4 + r];
                pass1_fwd(u, wy, wx);
            }
#pragma unroll
            for (int rho = 0; rho < 2; ++rho) {
                x1_write(u, rho, t, wbuf);
                __syncwarp();
                x1_read(u, rho, t, wbuf);
                __syncwarp();
            }
            pass2<false>(u);
            park<0, 32>(u, v ? slot1 : slot0);
        }
        VPROF(0)
        tmem_wait_st();
        __syncthreads();                    // exchange 1 is done everywhere: its buffers become the exchange-2 buffer
        x2_round(0, w, t, slot0, slot1, xb2);
        x2_round(1, w, t, slot0, slot1, xb2);
        VPROF(1)
        // ---- pass 3 and |F|^2 for the other modes of the view ----
        float4 *mine = a.sbuf + (((size_t)par * nslots + slot) * 8) * RNT + tid;
        if (M > 1) {
#pragma unroll 1
            for (int v = 0; v < 2; ++v) {
                float2 u[32];
                fetch<0, 32>(u, v ? slot1 : slot0);
                tmem_wait_ld();
                pass3<false>(u);
#pragma unroll
                for (int j = 0; j < 8; ++j)
                    mine[j * RNT + 256 * v] = make_float4(abs2_rn(u[4 * j]), abs2_rn(u[4 * j + 1]), abs2_rn(u[4 * j + 2]), abs2_rn(u[4 * j + 3]));
                park<0, 32>(u, v ? slot1 : slot0);
            }
            VPROF(2)
            tmem_wait_st();
            __syncthreads();
            if (tid == 0 && alive) {
                __threadfence();
                atomicAdd(a.gbar + cl, 1);
                const int want = M * (it + 1);
                int vv, spins = 0;
                do {
                    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];\n" : "=r"(vv) : "l"(a.gbar + cl) : "memory");
                } while (vv < want && ++spins < SPIN_LIMIT);
                if (vv < want) alive = false;
            }
            __syncthreads();
        }
        VPROF(3)
        // ---- S4 (eq. (4)) and the first inverse pass ----
#pragma unroll 1
        for (int v = 0; v < 2; ++v) {
            float2 u[32];
            fetch<0, 32>(u, v ? slot1 : slot0);
            tmem_wait_ld();
            if (M == 1) pass3<false>(u);
            const int vtid = 256 * v + tid;
            const float4 *ampv = reinterpret_cast<const float4 *>(a.amp + (size_t)view * RNN) + vtid;
            const float4 *peers = a.sbuf + (((size_t)par * nslots + (size_t)cl * M) * 8) * RNT + vtid;
            constexpr int JB = (MT == 1 || MT == 2) ? 4 : 1;
            constexpr int MP = MT ? MT : 8;
#pragma unroll
            for (int j0 = 0; j0 < 8; j0 += JB) {
                float4 pv[MP][JB], am[JB];
#pragma unroll
                for (int jj = 0; jj < JB; ++jj) am[jj] = __ldg(ampv + (j0 + jj) * RNT);
#pragma unroll
                for (int mm = 0; mm < MP; ++mm)
                    if (mm < M && mm != m) {
#pragma unroll
                        for (int jj = 0; jj < JB; ++jj) pv[mm][jj] = __ldcg(peers + ((size_t)mm * 8 + j0 + jj) * RNT);
                    }
#pragma unroll
                for (int jj = 0; jj < JB; ++jj) {
                    const int j = j0 + jj;
                    float4 S = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
                    for (int mm = 0; mm < MP; ++mm) {
                        if (mm < M) {
                            float4 x;
                            if (mm == m) x = make_float4(abs2_rn(u[4 * j]), abs2_rn(u[4 * j + 1]), abs2_rn(u[4 * j + 2]), abs2_rn(u[4 * j + 3]));
                            else x = pv[mm][jj];
                            S.x += x.x; S.y += x.y; S.z += x.z; S.w += x.w;
                        }
                    }
                    const float Sv[4] = {S.x, S.y, S.z, S.w}, av[4] = {am[jj].x, am[jj].y, am[jj].z, am[jj].w};
#pragma unroll
                    for (int cc = 0; cc < 4; ++cc) {
                        const float rs = rsqrtf(Sv[cc] + a.eps);
                        const float d = Sv[cc] * rs - av[cc];
                        e0 = fmaf(d, d, e0);
                        e1 = fmaf(av[cc], av[cc], e1);
                        const float sc = av[cc] * rs * cfac;
                        u[4 * j + cc].x *= sc;
                        u[4 * j + cc].y *= sc;
                    }
                }
            }
            pass3<true>(u);
            park<0, 32>(u, v ? slot1 : slot0);
        }
        VPROF(4)
        tmem_wait_st();
        x2_round(0, w, t, slot0, slot1, xb2);
        x2_round(1, w, t, slot0, slot1, xb2);
        VPROF(5)
        // ---- rest of the inverse FFT and S6: psi_new = psi_old + beta (G - P O) ----
#pragma unroll 1
        for (int v = 0; v < 2; ++v) {
            const int vw = 8 * v + w;
            const float2 *Pk = Pfr + vw * RN + t, *Ow = Ofr + (size_t)vw * a.W + t;
            float2 *ps = frame + vw * RN + t;
            float2 u[32];
            fetch<0, 32>(u, v ? slot1 : slot0);
            tmem_wait_ld();
            pass2<true>(u);
#pragma unroll
            for (int rho = 0; rho < 2; ++rho) {
                x1_write(u, rho, t, wbuf);
                __syncwarp();
                x1_read(u, rho, t, wbuf);
                __syncwarp();
            }
            {
                float2 wy[8], wx[4];
#pragma unroll
                for (int q = 0; q < 8; ++q) wy[q] = s_wy[vw * 8 + q];
#pragma unroll
                for (int r = 0; r < 4; ++r) wx[r] = s_wx[t * 4 + r];
                pass1_inv(u, wy, wx);
            }
#pragma unroll
            for (int h = 0; h < 4; ++h) {
                float2 pp[8], o[8], old[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const int ee = 8 * h + e;
                    pp[e] = __ldg(Pk + (ee >> 2) * 16 * RN + (ee & 3) * 32);
                    o[e] = __ldg(Ow + (size_t)(ee >> 2) * 16 * a.W + (ee & 3) * 32);
                    old[e] = ld_l2hint(ps + (ee >> 2) * 16 * RN + (ee & 3) * 32, drop);
                }
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const int ee = 8 * h + e;
                    const float2 po = cmul(pp[e], o[e]);
                    const float tx = u[ee].x - po.x, ty = u[ee].y - po.y;
                    const float2 nw = make_float2(fmaf(a.beta, tx, old[e].x), fmaf(a.beta, ty, old[e].y));
                    e2 = fmaf(tx, tx, fmaf(ty, ty, e2));
                    e3 = fmaf(nw.x, nw.x, fmaf(nw.y, nw.y, e3));
                    __stcs(ps + (ee >> 2) * 16 * RN + (ee & 3) * 32, nw);
                }
            }
        }
        VPROF(6)
    }
#ifdef DM_VT_PROF
    if (tid == 0 && (blockIdx.x == 0 || blockIdx.x == 1 || blockIdx.x == 151) && it > 0)
        printf("blk %d it %d: SEG_A %lld | x2 fwd %lld | p3+publish %lld | gbar %lld | S4+p3i %lld | x2 inv %lld | SEG_C %lld (cycles per frame)\n", blockIdx.x, it,
               prof[0] / it, prof[1] / it, prof[2] / it, prof[3] / it, prof[4] / it, prof[5] / it, prof[6] / it);
#endif
    asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
    __syncthreads();
    if (w == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" :: "r"(s_tmem), "r"(256) : "memory");
    float acc[4] = {m == 0 ? e0 : 0.f, m == 0 ? e1 : 0.f, e2 * a.beta * a.beta, e3};
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int s = 16; s > 0; s >>= 1) acc[i] += __shfl_xor_sync(0xffffffffu, acc[i], s);
    if (t == 0)
#pragma unroll
        for (int i = 0; i < 4; ++i) red[i * 8 + w] = acc[i];
    __syncthreads();
    if (tid < 4) {
        float s = 0.f;
        for (int ww = 0; ww < 8; ++ww) s += red[tid * 8 + ww];
        a.part[(size_t)blockIdx.x * 4 + tid] = s;
    }
}

} // namespace dmvt
#endif // __CUDACC__
