// dm_pairfft.cuh -- path 5: the register-resident 128 x 128 frame transform of dm_regfft.cuh with the
// frame split over a CLUSTER OF TWO CTAs of 256 threads, two CTAs (of different frames) per SM.
// Steps S1-S6 of DESIGN.md; eqs. (2)-(4) of arXiv:1808.10375.
//
// Why: with one 512-thread CTA per SM (path 3) the memory-side phases of a frame (S1: P, O, psi in; S4: the
// |F|^2 exchange between the modes of a view; S6: psi out) and the FFT passes run strictly one after another.
// Two independent CTAs per SM overlap them: while one waits for L2 / the group barrier / its stores, the other
// one's FFT passes keep the FP32 pipe busy.
//
// How: CTA c (cluster rank 0 / 1) runs the "virtual warps" 8 c .. 8 c + 7 of dm_regfft.cuh's 16-warp
// schedule, with the same register layouts, passes, twiddles and spectrum layout (so sqrt(I) is stored exactly
// as for path 3).  Pass 1, exchange 1 (a transpose inside each warp) and pass 2 never leave a warp.  Exchange 2
// ((warp w, reg 16 z + c') <-> (warp c', reg 16 z + w)) moves half of every thread's registers to the other CTA:
// those elements are written straight into the peer's shared memory (DSMEM, st.async) and counted on an mbarrier
// of the receiving CTA; the hardware cluster barrier (relaxed arrive) only says "my buffer may be overwritten".  Everything else is CTA-local:
//   registers     32 complex per thread (half a frame per CTA)
//   tensor memory 256 columns per CTA: psi_old and P*O of the half frame, parked during the FFTs
//   shared memory 64 KiB prefetch buffer (next half frame of psi by cp.async.bulk; sqrt(I) of this view takes
//                 over its first half once S1 has read it) + 36 KiB exchange buffer + twiddles
// The M = K*L frames of a view sit on M consecutive clusters; their |F|^2 go through L2 (sbuf) behind a
// release / acquire counter (all CTAs are resident: the grid is sized from cudaOccupancyMaxActiveClusters).
#pragma once
#include "dm_regfft.cuh"

#ifdef __CUDACC__
namespace dmpair {

using namespace dmreg;

constexpr int PNT = 256;                         // threads per CTA
constexpr int P_PBUF = 65536;                    // prefetch buffer: half a frame of psi
constexpr int P_XBUF = 8 * X1_WARP;              // 36 864 B >= 32 KiB of one exchange-2 round
constexpr int PAIR_SMEM = P_PBUF + P_XBUF + 2048;
constexpr int SPIN_LIMIT = 1 << 22;              // group barrier polls before a CTA gives up (no hang on a mis-sized grid)

__device__ __forceinline__ void mbar_expect(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n"
                 :: "r"((uint32_t)__cvta_generic_to_shared(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_copy(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n"
                 :: "r"((uint32_t)__cvta_generic_to_shared(dst_smem)), "l"(src_gmem), "r"(bytes),
                    "r"((uint32_t)__cvta_generic_to_shared(bar)) : "memory");
}
__device__ __forceinline__ uint32_t cluster_rank()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;\n" : "=r"(r));
    return r;
}
__device__ __forceinline__ uint32_t map_peer(uint32_t smem_addr, uint32_t rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;\n" : "=r"(r) : "r"(smem_addr), "r"(rank));
    return r;
}
// 8-byte store into (possibly the peer's) shared memory that reports its bytes to an mbarrier of the SAME CTA as
// the destination: the receiver waits on its own barrier, no fence and no cluster barrier on the data path
__device__ __forceinline__ void st_async(uint32_t addr, float2 v, uint32_t bar)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.f32 [%0], {%1, %2}, [%3];\n"
                 :: "r"(addr), "f"(v.x), "f"(v.y), "r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect(uint64_t *bar, uint32_t bytes) { mbar_expect(bar, bytes); }
__device__ __forceinline__ void mbar_wait_cluster(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAITC_%=:\n"
        "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONEC_%=;\n"
        "bra WAITC_%=;\n"
        "DONEC_%=:\n"
        "}\n" :: "r"((uint32_t)__cvta_generic_to_shared(bar)), "r"(parity) : "memory");
}
// "my exchange buffer may be overwritten": no data is published, so no fence (a .release arrive costs a MEMBAR
// that waits for every store in flight, the psi stores of S6 included)
__device__ __forceinline__ void cluster_arrive_relaxed()
{
    __threadfence_block();          // the reads of the buffer have been performed (a bare relaxed arrive was observed to overtake them)
    asm volatile("barrier.cluster.arrive.relaxed.aligned;\n" ::: "memory");
}

// psi rows of the half frame of cluster rank c: y = 8 c + w + 16 i (w < 8, i < 8); in the prefetch buffer
// row (i, w) sits at (8 i + w) * 1 KiB.  Half A = i < 4, half B = i >= 4: four 8 KiB copies each.
__device__ __forceinline__ void load_psi_half(unsigned char *pbuf, const unsigned char *frame, int c, int half, uint64_t *bar)
{
    mbar_expect(bar, 32768);
#pragma unroll
    for (int i = 4 * half; i < 4 * half + 4; ++i)
        bulk_copy(pbuf + i * 8192, frame + (size_t)(16 * i + 8 * c) * RN * sizeof(float2), 8192, bar);
}
// sqrt(I) of the view in the spectrum layout [j][virtual tid][4]: this CTA's 256 threads own 4 KiB of every j
__device__ __forceinline__ void load_amp_half(unsigned char *pbuf, const float *amp_view, int c, uint64_t *bar)
{
    mbar_expect(bar, 32768);
#pragma unroll
    for (int j = 0; j < 8; ++j)
        bulk_copy(pbuf + j * 4096, amp_view + ((size_t)j * RNT + 256 * c) * 4, 4096, bar);
}

// exchange 2 for one z: this thread's registers 16 z + c' go to virtual warp c' (CTA c' >> 3), slot
// ((c' & 7) 16 + vw) 32 + lane of that CTA's buffer.  The half that stays goes by st.shared, the half that leaves by
// st.async into the peer's buffer, counted on the peer's barrier; then every warp arrives on its OWN CTA's barrier
// and announces the 2 KiB that the peer's same-numbered warp sends.
__device__ __forceinline__ void x2_write_pair(const float2 (&u)[32], int z, int c, int vw, int t, float2 *own, uint32_t peer,
                                              uint32_t peer_bar, uint64_t *own_bar)
{
    float2 *lp = own + vw * 32 + t;
    const uint32_t rp = peer + (uint32_t)(vw * 32 + t) * 8u;
    // registers 16 z + 8 c + i stay (c' = 8 c + i), registers 16 z + 8 (1 - c) + i leave
#define DM_X2_ROUND(STAY, LEAVE)                                                    \
    {                                                                               \
        _Pragma("unroll") for (int i = 0; i < 8; ++i) st_async(rp + i * 4096, u[LEAVE + i], peer_bar); \
        _Pragma("unroll") for (int i = 0; i < 8; ++i) lp[i * 512] = u[STAY + i];    \
    }
    if (z == 0) {
        if (c == 0) DM_X2_ROUND(0, 8) else DM_X2_ROUND(8, 0)
    } else {
        if (c == 0) DM_X2_ROUND(16, 24) else DM_X2_ROUND(24, 16)
    }
#undef DM_X2_ROUND
    __syncwarp();
    if (t == 0) mbar_arrive_expect(own_bar, 2048);
}

#ifdef DM_PAIR_PROF
#define PROF_T(i) { const long long now_ = clock64(); prof[i] += now_ - tprev; tprev = now_; }
#else
#define PROF_T(i)
#endif

struct PairArgs {
    int n_views, K, L, H, W;
    const int2 *pos;
    const float2 *P, *O;
    float2 *psi;
    const float *amp;
    const float2 *wy, *wx;
    float4 *sbuf;               // [2][frames in flight][8][512]  |F|^2 of every resident frame (mode-sum exchange, L2)
    float *part;                // [grid][4]
    float beta, eps;
    int *gbar;                  // [groups] arrival counters of the 2 M CTAs of a view
    int *gave_up;               // sticky flag: set when a CTA stops waiting at the group barrier (dm_get_errors reports it)
};

// grid = 2 * (frames in flight); cluster (2,1,1); frame slot f = blockIdx.x / 2 holds mode f % M of the
// view group f / M; group g processes views g, g + n_groups, ...
template <int MT>
__global__ void __launch_bounds__(PNT, 2) pairfft128_kernel(const PairArgs a)
{
    extern __shared__ __align__(128) unsigned char smem[];
    unsigned char *pbuf = smem;
    unsigned char *xbuf = smem + P_PBUF;
    float2 *s_wy = reinterpret_cast<float2 *>(smem + P_PBUF + P_XBUF);
    float2 *s_wx = s_wy + 128;
    __shared__ float red[4 * 8];
    __shared__ uint32_t s_tmem;
    __shared__ __align__(8) uint64_t mb_lo, mb_hi, mb_amp, mb_x;     // mb_x: one phase per exchange-2 round

    const int tid = threadIdx.x, w = tid >> 5, t = tid & 31;
    const int c = (int)cluster_rank();
    const int vw = 8 * c + w, vtid = 256 * c + tid;
    const int M = MT ? MT : a.K * a.L;
    const int slot = blockIdx.x >> 1, nslots = gridDim.x >> 1;
    const int m = slot % M, cl = slot / M, ncl = nslots / M;
    const int k = m / a.L, l = m % a.L;
    if (tid < 128) s_wy[tid] = a.wy[tid];
    else s_wx[tid - 128] = a.wx[tid - 128];
    if (tid == 0) {
        mbar_init(&mb_lo, 1);
        mbar_init(&mb_hi, 1);
        mbar_init(&mb_amp, 1);
        mbar_init(&mb_x, 8);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    if (w == 0) {       // half of the SM's tensor memory (two CTAs per SM)
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n"
                     :: "r"((uint32_t)__cvta_generic_to_shared(&s_tmem)), "r"(256) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
    cluster_arrive();
    cluster_wait();                 // both CTAs are running (their shared memory may be written from now on)
    asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
    const uint32_t t_psi = s_tmem + ((uint32_t)(32 * (w & 3)) << 16) + (uint32_t)(w >> 2) * 128u;
    const uint32_t t_po = t_psi + 64u;

    unsigned char *wbuf = xbuf + w * X1_WARP;
    float2 *xb2 = reinterpret_cast<float2 *>(xbuf);
    const uint32_t xb_peer = map_peer((uint32_t)__cvta_generic_to_shared(xbuf), (uint32_t)(c ^ 1));
    const uint32_t bar_peer = map_peer((uint32_t)__cvta_generic_to_shared(&mb_x), (uint32_t)(c ^ 1));
    int xpar = 0;
    const float2 *Pk = a.P + (size_t)k * RNN + vw * RN + t;
    const float cfac = a.beta > 0.f ? 1.f / (float)RNN : 0.f;
    float e0 = 0.f, e1 = 0.f, e2 = 0.f, e3 = 0.f;
    int par = 0;
    bool alive = true;
    if (tid == 0 && cl < ncl && cl < a.n_views) {
        const unsigned char *src = reinterpret_cast<const unsigned char *>(a.psi + ((size_t)cl * M + m) * RNN);
        load_psi_half(pbuf, src, c, 0, &mb_lo);
        load_psi_half(pbuf, src, c, 1, &mb_hi);
    }

#ifdef DM_PAIR_PROF
    long long prof[12] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0}, tprev = clock64();
    unsigned long long g0, g1;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g0));
    const long long c_loop0 = tprev;
#endif
    int it = 0;
    for (int view = cl; cl < ncl && view < a.n_views; view += ncl, par ^= 1, ++it) {
        const int2 p0 = a.pos[view];
        float2 *psi_f = a.psi + ((size_t)view * M + m) * RNN + vw * RN + t;
        const float2 *Ow = a.O + (size_t)l * a.H * a.W + (size_t)(p0.x + vw) * a.W + p0.y + t;
        const int nview = view + ncl;
        const unsigned char *nsrc = reinterpret_cast<const unsigned char *>(a.psi + ((size_t)nview * M + m) * RNN);
        float2 u[32];
        // ---- S1 + S2: R = 2 P O - psi; psi_old and P*O parked in tensor memory ----
        {
            float2 po[32], o[16];
#pragma unroll
            for (int e = 0; e < 32; ++e) po[e] = __ldg(Pk + (e >> 2) * 16 * RN + (e & 3) * 32);
#pragma unroll
            for (int e = 0; e < 16; ++e) o[e] = __ldg(Ow + (size_t)(e >> 2) * 16 * a.W + (e & 3) * 32);
            mbar_wait(&mb_lo, par);
            mbar_wait(&mb_hi, par);
            const float2 *ps = reinterpret_cast<const float2 *>(pbuf) + w * RN + t;
#pragma unroll
            for (int e = 0; e < 16; ++e) po[e] = cmul(po[e], o[e]);
#pragma unroll
            for (int e = 0; e < 16; ++e) o[e] = __ldg(Ow + (size_t)((e + 16) >> 2) * 16 * a.W + (e & 3) * 32);
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                if (h == 1) {
#pragma unroll
                    for (int e = 0; e < 16; ++e) po[16 + e] = cmul(po[16 + e], o[e]);
                }
#pragma unroll
                for (int i = 4 * h; i < 4 * h + 4; ++i) {
#pragma unroll
                    for (int r = 0; r < 4; ++r) u[4 * i + r] = ps[i * 8 * RN + r * 32];
                    tmem_st8(t_psi + 8 * i, u[4 * i], u[4 * i + 1], u[4 * i + 2], u[4 * i + 3]);
                    tmem_st8(t_po + 8 * i, po[4 * i], po[4 * i + 1], po[4 * i + 2], po[4 * i + 3]);
#pragma unroll
                    for (int r = 0; r < 4; ++r)
                        u[4 * i + r] = make_float2(2.f * po[4 * i + r].x - u[4 * i + r].x, 2.f * po[4 * i + r].y - u[4 * i + r].y);
                }
            }
        }
        __syncthreads();                    // the whole prefetch buffer has been read
        PROF_T(0)
        if (tid == 0) {
            load_amp_half(pbuf, a.amp + (size_t)view * RNN, c, &mb_amp);
            if (nview < a.n_views) load_psi_half(pbuf, nsrc, c, 1, &mb_hi);
        }
        tmem_wait_st();
        // ---- S3: forward 2-D FFT ----
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
        cluster_arrive_relaxed();           // this CTA's exchange buffer is free (exchange 1 is done)
        pass2<false>(u);
        PROF_T(1)
#pragma unroll
        for (int z = 0; z < 2; ++z) {
            cluster_wait();                 // ... and so is the peer's
            x2_write_pair(u, z, c, vw, t, xb2, xb_peer, bar_peer, &mb_x);
            mbar_wait_cluster(&mb_x, xpar); // both halves of the round have landed
            xpar ^= 1;
            x2_read(u, z, w, t, xb2);
            if (z == 0) cluster_arrive_relaxed();   // read: free for the next round
        }
        PROF_T(2)
        pass3<false>(u);
        // ---- S4: mode-summed modulus constraint (|F|^2 exchanged through L2) ----
        {
            float4 *mine = a.sbuf + (((size_t)par * nslots + slot) * 8) * RNT + vtid;
            if (M > 1) {
#pragma unroll
                for (int j = 0; j < 8; ++j)
                    mine[j * RNT] = make_float4(abs2_rn(u[4 * j]), abs2_rn(u[4 * j + 1]), abs2_rn(u[4 * j + 2]), abs2_rn(u[4 * j + 3]));
                PROF_T(3)
                __syncthreads();
                if (tid == 0 && alive) {
                    __threadfence();
                    atomicAdd(a.gbar + cl, 1);
                    const int want = 2 * M * (it + 1);
                    int v, spins = 0;
                    do {
                        asm volatile("ld.acquire.gpu.global.s32 %0, [%1];\n" : "=r"(v) : "l"(a.gbar + cl) : "memory");
                    } while (v < want && ++spins < SPIN_LIMIT);
                    if (v < want) { alive = false; atomicExch(a.gave_up, 1); }
                }
                __syncthreads();
            }
            PROF_T(4)
            mbar_wait(&mb_amp, par);
            const float4 *ampv = reinterpret_cast<const float4 *>(pbuf) + tid;
            const float4 *peers = a.sbuf + (((size_t)par * nslots + (size_t)cl * M) * 8) * RNT + vtid;
            constexpr int JB = (MT == 1 || MT == 2) ? 4 : 1;
            constexpr int MP = MT ? MT : 8;
#pragma unroll
            for (int j0 = 0; j0 < 8; j0 += JB) {
                float4 pv[MP][JB];
#pragma unroll
                for (int mm = 0; mm < MP; ++mm)
                    if (mm < M && mm != m) {
#pragma unroll
                        for (int jj = 0; jj < JB; ++jj) pv[mm][jj] = __ldcg(peers + ((size_t)mm * 8 + j0 + jj) * RNT);
                    }
#pragma unroll
                for (int jj = 0; jj < JB; ++jj) {
                    const int j = j0 + jj;
                    const float4 am = ampv[j * PNT];
                    float4 S = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
                    for (int mm = 0; mm < MP; ++mm) {
                        if (mm < M) {
                            float4 v;
                            if (mm == m) v = make_float4(abs2_rn(u[4 * j]), abs2_rn(u[4 * j + 1]), abs2_rn(u[4 * j + 2]), abs2_rn(u[4 * j + 3]));
                            else v = pv[mm][jj];
                            S.x += v.x; S.y += v.y; S.z += v.z; S.w += v.w;
                        }
                    }
                    const float Sv[4] = {S.x, S.y, S.z, S.w}, av[4] = {am.x, am.y, am.z, am.w};
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
        }
        // ---- S5: inverse 2-D FFT (mirror) ----
        PROF_T(5)
        cluster_arrive_relaxed();           // exchange buffer read, sqrt(I) (prefetch half A) consumed
        pass3<true>(u);
        PROF_T(6)
#pragma unroll
        for (int z = 0; z < 2; ++z) {
            cluster_wait();                 // both buffers free; every thread of the pair is past S4
            if (z == 0 && tid == 0 && nview < a.n_views) load_psi_half(pbuf, nsrc, c, 0, &mb_lo);
            x2_write_pair(u, z, c, vw, t, xb2, xb_peer, bar_peer, &mb_x);
            mbar_wait_cluster(&mb_x, xpar);
            xpar ^= 1;
            x2_read(u, z, w, t, xb2);
            if (z == 0) cluster_arrive_relaxed();
        }
        PROF_T(7)
        pass2<true>(u);
        __syncthreads();                    // every warp has read its part of the exchange-2 buffer
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
        PROF_T(8)
        // ---- S6: psi_new = psi_old + beta (G - P O) ----
#pragma unroll
        for (int i = 0; i < 8; i += 2) {
            float2 old[8], po[8];
            tmem_ld8(t_psi + 8 * i, old[0], old[1], old[2], old[3]);
            tmem_ld8(t_psi + 8 * i + 8, old[4], old[5], old[6], old[7]);
            tmem_ld8(t_po + 8 * i, po[0], po[1], po[2], po[3]);
            tmem_ld8(t_po + 8 * i + 8, po[4], po[5], po[6], po[7]);
            tmem_wait_ld();
#pragma unroll
            for (int r = 0; r < 8; ++r) {
                const int e = 4 * i + r;
                const float tx = u[e].x - po[r].x, ty = u[e].y - po[r].y;
                const float2 nw = make_float2(fmaf(a.beta, tx, old[r].x), fmaf(a.beta, ty, old[r].y));
                e2 = fmaf(tx, tx, fmaf(ty, ty, e2));
                e3 = fmaf(nw.x, nw.x, fmaf(nw.y, nw.y, e3));
                psi_f[(e >> 2) * 16 * RN + (e & 3) * 32] = nw;
            }
        }
        PROF_T(9)
    }
#ifdef DM_PAIR_PROF
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g1));
    if (tid == 0 && (blockIdx.x == 0 || blockIdx.x == 1 || blockIdx.x == 151 || blockIdx.x == 295))
        printf("blk %d start %llu ns end %llu ns loop cycles %lld\n", blockIdx.x, g0 % 100000000ull, g1 % 100000000ull, clock64() - c_loop0);
    if (tid == 0 && (blockIdx.x == 0 || blockIdx.x == 1 || blockIdx.x == 151))
        printf("blk %d it %d: S1 %lld | p1+x1 %lld | p2+x2 %lld | p3+sbuf %lld | gbar %lld | S4 %lld | p3i %lld | x2i %lld | p2i+x1+p1i %lld | S6 %lld  (cycles per frame)\n", blockIdx.x, it,
               prof[0] / it, prof[1] / it, prof[2] / it, prof[3] / it, prof[4] / it, prof[5] / it, prof[6] / it, prof[7] / it, prof[8] / it, prof[9] / it);
#endif
    asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
    cluster_arrive();
    cluster_wait();                         // no CTA leaves while its peer may still write to it
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

} // namespace dmpair
#endif // __CUDACC__
