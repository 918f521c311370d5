// dm_regfft.cuh -- register-resident 128 x 128 frame transform of the psi update (steps S1-S6
// of DESIGN.md; eqs. (2)-(4) of arXiv:1808.10375).  Included by dm_kernels.cuh.
//
// One CTA of 512 threads holds ONE whole 128 x 128 complex64 mode frame in registers (32
// elements per thread).  The 2-D FFT is three register passes with two shared-memory exchanges:
//
//   L0 (load/store layout, coalesced rows):  thread (warp w, lane t), register a = 4 i + r
//        holds pixel  y = w + 16 i (i < 8),  x = t + 32 r (r < 4)
//   pass 1   radix-8 along y over i  (-> q),   twiddle w128^(w q)
//            radix-4 along x over r  (-> r'),  twiddle w128^(t r')          register a' = 4 q + r'
//   exch. 1  32 x 32 transpose inside each warp: (lane t, reg a') -> (lane a', reg t)
//   pass 2   radix-32 along x over t (-> c):   kx = r' + 4 c               x is finished
//   exch. 2  16 x 16 transpose across the warps, lane fixed, the register bit z = c >> 4 stays:
//            (warp w, reg 16 z + c') -> (warp c', reg 16 z + w)
//   pass 3   radix-16 along y over w (-> k2):  ky = q + 8 k2               y is finished
//
//   spectrum layout: thread (warp w', lane t' = 4 q + r'), register e = 16 z + k2 holds
//        F[ky = q + 8 k2][kx = r' + 4 (w' + 16 z)]
//
// The inverse runs the mirrored passes (both exchanges are involutions), ending in L0.  The
// Fourier-modulus step (eq. (4)) is pointwise, so it runs in the spectrum layout; sqrt(I) is
// stored once in that layout (spec_index table, dm_set_data).
//
// Every function here is __host__ __device__: tests run exactly this code on the CPU through
// dm_host_fft2 (512 emulated threads, phase by phase) before anything goes to a GPU.
#pragma once
#include <cuda_runtime.h>

#include "dm_fft.cuh"

namespace dmreg {

using namespace dmfft;

constexpr int RN = 128, RNN = RN * RN, RNT = 512, REPT = 32;
// exchange buffer: 16 warps x (2 blocks of 16 rows x 144 B) for exchange 1, 64 KiB for exchange 2
constexpr int X1_ROW = 144;                                                     // bytes
// path 3 keeps a warp's exchange-1 rows inside the 4 KiB that the same warp reads in exchange 2 (rows 0..27) plus a
// private spare strip behind the 64 KiB (rows 28..31), so exchange 1 never touches what another warp still has to
// read: no block barrier between exchange 2 and exchange 1.  Spare strips start at 64 (mod 128) bytes: the 128-bit
// loads of rows 24..27 (main) and 28..31 (spare) then fall on disjoint banks.
constexpr int X1S_MAIN_ROWS = 28, X1S_SPARE = 640, X1S_SPARE_OFF = 65536 + 64;
constexpr int XBUF3_BYTES = X1S_SPARE_OFF + 16 * X1S_SPARE;                       // 75840

// cos / sin of 2 pi m / 32
__device__ __host__ constexpr float c32(int m)
{
    constexpr float C[32] = {1.f, 0.98078528040323043f, 0.92387953251128674f, 0.83146961230254524f, 0.70710678118654757f,
        0.55557023301960229f, 0.38268343236508984f, 0.19509032201612833f, 0.f, -0.19509032201612819f, -0.38268343236508973f,
        -0.55557023301960196f, -0.70710678118654746f, -0.83146961230254535f, -0.92387953251128674f, -0.98078528040323043f,
        -1.f, -0.98078528040323043f, -0.92387953251128685f, -0.83146961230254546f, -0.70710678118654768f,
        -0.55557023301960218f, -0.38268343236509034f, -0.19509032201612866f, 0.f, 0.1950903220161283f, 0.38268343236509f,
        0.55557023301960184f, 0.70710678118654735f, 0.83146961230254524f, 0.92387953251128652f, 0.98078528040323032f};
    return C[m & 31];
}
__device__ __host__ constexpr float s32(int m) { return c32(m - 8); }

// a * w32^M (forward: exp(-2 pi i M/32); inverse: conjugate), M a compile-time constant
template <bool INV, int M> DM_HD float2 mul_w32(float2 a)
{
    constexpr int m = M & 31;
    if (m == 0) return a;
    if (m == 16) return make_float2(-a.x, -a.y);
    if (m == 8) return mul_mi<INV>(a);
    if (m == 24) return mul_mi<!INV>(a);
    constexpr float c = c32(m), s = s32(m);
    return INV ? make_float2(a.x * c - a.y * s, a.x * s + a.y * c)
               : make_float2(a.x * c + a.y * s, a.y * c - a.x * s);
}

// natural-order 32-point DFT in registers: n = 8 n1 + n2, k = k1 + 4 k2
template <bool INV> DM_HD void dft32(float2 (&x)[32])
{
#pragma unroll
    for (int n2 = 0; n2 < 8; ++n2) dft4<INV>(x[n2], x[8 + n2], x[16 + n2], x[24 + n2]);   // -> x[8 k1 + n2]
#define DM_TW(K1, N2) x[8 * K1 + N2] = mul_w32<INV, K1 * N2>(x[8 * K1 + N2]);
#define DM_TWROW(K1) DM_TW(K1, 1) DM_TW(K1, 2) DM_TW(K1, 3) DM_TW(K1, 4) DM_TW(K1, 5) DM_TW(K1, 6) DM_TW(K1, 7)
    DM_TWROW(1) DM_TWROW(2) DM_TWROW(3)
#undef DM_TWROW
#undef DM_TW
    float2 y[32];
#pragma unroll
    for (int k1 = 0; k1 < 4; ++k1) {
        float2 v[8];
#pragma unroll
        for (int n2 = 0; n2 < 8; ++n2) v[n2] = x[8 * k1 + n2];
        dft8<INV>(v);
#pragma unroll
        for (int k2 = 0; k2 < 8; ++k2) y[k1 + 4 * k2] = v[k2];
    }
#pragma unroll
    for (int k = 0; k < 32; ++k) x[k] = y[k];
}

// ---- register passes ------------------------------------------------------------------
// wy[q] = w128^(w q) (q < 8, per warp), wx[r'] = w128^(t r') (r' < 4, per lane); forward sign.
DM_HD void pass1_fwd(float2 (&u)[32], const float2 *wy, const float2 *wx)
{
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        float2 v[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) v[i] = u[4 * i + r];
        dft8<false>(v);
        u[r] = v[0];
#pragma unroll
        for (int q = 1; q < 8; ++q) u[4 * q + r] = cmul(v[q], wy[q]);
    }
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        dft4<false>(u[4 * q], u[4 * q + 1], u[4 * q + 2], u[4 * q + 3]);
#pragma unroll
        for (int rp = 1; rp < 4; ++rp) u[4 * q + rp] = cmul(u[4 * q + rp], wx[rp]);
    }
}

DM_HD void pass1_inv(float2 (&u)[32], const float2 *wy, const float2 *wx)
{
#pragma unroll
    for (int q = 0; q < 8; ++q) {
#pragma unroll
        for (int rp = 1; rp < 4; ++rp) u[4 * q + rp] = cmulc(u[4 * q + rp], wx[rp]);
        dft4<true>(u[4 * q], u[4 * q + 1], u[4 * q + 2], u[4 * q + 3]);
    }
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        float2 v[8];
        v[0] = u[r];
#pragma unroll
        for (int q = 1; q < 8; ++q) v[q] = cmulc(u[4 * q + r], wy[q]);
        dft8<true>(v);
#pragma unroll
        for (int i = 0; i < 8; ++i) u[4 * i + r] = v[i];
    }
}

template <bool INV> DM_HD void pass2(float2 (&u)[32]) { dft32<INV>(u); }

// pass 3 works on the two register halves z = 0, 1 independently (they are also the two rounds of exchange 2)
template <bool INV> DM_HD void pass3_half(float2 (&u)[32], int z)
{
    float2 v[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = u[16 * z + i];
    dft16<INV>(v);
#pragma unroll
    for (int i = 0; i < 16; ++i) u[16 * z + i] = v[i];
}
template <bool INV> DM_HD void pass3(float2 (&u)[32])
{
#pragma unroll
    for (int z = 0; z < 2; ++z) {
        float2 v[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) v[i] = u[16 * z + i];
        dft16<INV>(v);
#pragma unroll
        for (int i = 0; i < 16; ++i) u[16 * z + i] = v[i];
    }
}

// ---- exchange 1: 32 x 32 transpose inside a warp, two rounds of 16 registers ----------
// Round rho moves the elements (reg a', lane b) with (a' >> 4) == (b >> 4) ^ rho, so every lane
// writes 16 registers and reads 16 registers per round (4.5 KiB of buffer per warp).  Rows of
// 16 elements are padded to 144 B: 64-bit stores of a row and 128-bit loads down a column
// are both bank-conflict free.  The 32 rows of a warp are split over `mainp` (rows 0..27, inside
// the 4 KiB the warp itself reads in exchange 2) and `spare` (rows 28..31, its private strip).
DM_HD unsigned char *x1s_row(int r, unsigned char *mainp, unsigned char *spare)
{
    return r < X1S_MAIN_ROWS ? mainp + r * X1_ROW : spare + (r - X1S_MAIN_ROWS) * X1_ROW;
}
DM_HD void x1s_write(const float2 (&u)[32], int rho, int t, unsigned char *mainp, unsigned char *spare)
{
    const int h = (t >> 4) ^ rho;
    const int col = (t & 15) * 8;
    if (h == 0) {
#pragma unroll
        for (int j = 0; j < 16; ++j) *reinterpret_cast<float2 *>(mainp + j * X1_ROW + col) = u[j];
    } else {
#pragma unroll
        for (int j = 0; j < 16; ++j) *reinterpret_cast<float2 *>(x1s_row(16 + j, mainp, spare) + col) = u[16 + j];
    }
}
DM_HD void x1s_read(float2 (&u)[32], int rho, int t, unsigned char *mainp, unsigned char *spare)
{
    const int h = (t >> 4) ^ rho;
    const unsigned char *p = x1s_row(t, mainp, spare);
    if (h == 0) {
#pragma unroll
        for (int b = 0; b < 16; b += 2) {
            const float4 v = *reinterpret_cast<const float4 *>(p + b * 8);
            u[b] = make_float2(v.x, v.y);
            u[b + 1] = make_float2(v.z, v.w);
        }
    } else {
#pragma unroll
        for (int b = 0; b < 16; b += 2) {
            const float4 v = *reinterpret_cast<const float4 *>(p + b * 8);
            u[16 + b] = make_float2(v.x, v.y);
            u[16 + b + 1] = make_float2(v.z, v.w);
        }
    }
}

// ---- exchange 2: (warp w, reg 16 z + c') <-> (warp c', reg 16 z + w), lane fixed -------
// One round per z through a 64 KiB buffer: element (c', w, lane) at ((c' 16 + w) 32 + lane) 8 B.
DM_HD void x2_write(const float2 (&u)[32], int z, int w, int t, float2 *buf)
{
    float2 *p = buf + w * 32 + t;
    if (z == 0) {
#pragma unroll
        for (int c = 0; c < 16; ++c) p[c * 512] = u[c];
    } else {
#pragma unroll
        for (int c = 0; c < 16; ++c) p[c * 512] = u[16 + c];
    }
}

DM_HD void x2_read(float2 (&u)[32], int z, int w, int t, const float2 *buf)
{
    const float2 *p = buf + w * 512 + t;
    if (z == 0) {
#pragma unroll
        for (int i = 0; i < 16; ++i) u[i] = p[i * 32];
    } else {
#pragma unroll
        for (int i = 0; i < 16; ++i) u[16 + i] = p[i * 32];
    }
}

// storage position (float index inside a frame's N*N block) of register e of thread tid in the
// spectrum layout, as written with one float4 per 4 registers: [e >> 2][tid][e & 3]
DM_HD int spec_pos(int tid, int e) { return ((e >> 2) * RNT + tid) * 4 + (e & 3); }
// natural-order linear frequency index ky * 128 + kx that (tid, e) holds after the forward passes
DM_HD int spec_freq(int tid, int e)
{
    const int w = tid >> 5, t = tid & 31, q = t >> 2, rp = t & 3, z = e >> 4, k2 = e & 15;
    return (q + 8 * k2) * RN + rp + 4 * (w + 16 * z);
}
// L0 pixel (linear index y * 128 + x) of register a of thread tid
DM_HD int l0_pixel(int tid, int a)
{
    const int w = tid >> 5, t = tid & 31;
    return (w + 16 * (a >> 2)) * RN + t + 32 * (a & 3);
}

} // namespace dmreg

// =========================================================================================
// The kernel (device only)
// =========================================================================================
#ifdef __CUDACC__
#include <cooperative_groups.h>

namespace dmreg {

struct RegArgs {
    int n_views, K, L, H, W;
    const int2 *pos;            // (y0, x0) per view
    const float2 *P;            // [K][128][128]   current probe
    const float2 *O;            // [L][H][W]       current object
    float2 *psi;                // [n_views][K][L][128][128], updated in place
    const float *amp;           // [n_views][128*128] sqrt(I) in the spectrum layout (spec_pos)
    const float2 *wy;           // [16][8]  w128^(w q)
    const float2 *wx;           // [32][4]  w128^(t r')
    float4 *sbuf;               // [2][grid][8][512]  |F|^2 of every resident CTA (mode-sum exchange, L2)
    float *part;                // [grid][4]  (eF_num, eF_den, epsi_num, epsi_den) partial sums
    float beta, eps;
    int *gbar;                  // [grid / M] software group barrier counters (NULL: hardware cluster barrier)
};

// shared memory: [prefetch buffer 128 KiB | exchange buffer | twiddles 2 KiB]
// The prefetch buffer is filled by bulk asynchronous copies (TMA, cp.async.bulk) one step ahead:
//   half A (64 KiB): rows 0..63 of the next frame's psi, then -- once S1 has consumed them --
//                    sqrt(I) of the current view (consumed by S4), then the next psi rows again
//   half B (64 KiB): rows 64..127 of the next frame's psi
// so the HBM time of a frame hides behind the FFTs of the previous / current frame.
constexpr int PBUF_BYTES = 2 * 65536;
constexpr int REG_SMEM_V1 = PBUF_BYTES + XBUF3_BYTES + 2048;

__device__ __forceinline__ float abs2_rn(float2 f) { return __fmaf_rn(f.y, f.y, __fmul_rn(f.x, f.x)); }

// ---- tensor memory as a per-thread spill space ---------------------------------------------
// TMEM (256 KiB per SM, 128 lanes x 512 32-bit columns) is otherwise idle in this kernel (no
// tensor-core work).  The 32x32b shape maps lane i of a warp to TMEM lane 32 (warp % 4) + i, so a
// column range is private to a thread: psi_old and P*O of the frame (64 words each per thread)
// are parked there during the FFTs instead of being re-read from L2 / kept in shared memory.
__device__ __forceinline__ void tmem_st8(uint32_t taddr, float2 a, float2 b, float2 c, float2 d)
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};\n"
                 :: "r"(taddr), "r"(__float_as_uint(a.x)), "r"(__float_as_uint(a.y)), "r"(__float_as_uint(b.x)),
                    "r"(__float_as_uint(b.y)), "r"(__float_as_uint(c.x)), "r"(__float_as_uint(c.y)),
                    "r"(__float_as_uint(d.x)), "r"(__float_as_uint(d.y)) : "memory");
}
__device__ __forceinline__ void tmem_ld8(uint32_t taddr, float2 &a, float2 &b, float2 &c, float2 &d)
{
    uint32_t r0, r1, r2, r3, r4, r5, r6, r7;
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];\n"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3), "=r"(r4), "=r"(r5), "=r"(r6), "=r"(r7) : "r"(taddr) : "memory");
    a = make_float2(__uint_as_float(r0), __uint_as_float(r1));
    b = make_float2(__uint_as_float(r2), __uint_as_float(r3));
    c = make_float2(__uint_as_float(r4), __uint_as_float(r5));
    d = make_float2(__uint_as_float(r6), __uint_as_float(r7));
}
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;\n" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;\n" ::: "memory"); }
// ---- mbarrier + 1-D bulk copy (global -> this CTA's shared memory) ----------------------------
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" :: "r"((uint32_t)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" :: "r"((uint32_t)__cvta_generic_to_shared(bar)), "r"(parity) : "memory");
}
// one thread: announce `bytes` on the barrier and start the copy that will deliver them
__device__ __forceinline__ void bulk_load(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar)
{
    const uint32_t b = (uint32_t)__cvta_generic_to_shared(bar), d = (uint32_t)__cvta_generic_to_shared(dst_smem);
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" :: "r"(b), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n"
                 :: "r"(d), "l"(src_gmem), "r"(bytes), "r"(b) : "memory");
}
__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;\n" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;\n" ::: "memory"); }

// -DDM_REG_PROF (DM_NVCC_EXTRA of build.py): thread 0 of CTAs 0, 1 and 100 accumulates clock64 per phase and prints the
// mean cycles per frame at the end of the launch (the table of DESIGN.md 6.1; measurement builds only)
#ifdef DM_REG_PROF
#define RPROF(i) { const long long now_ = clock64(); prof[i] += now_ - tprev; tprev = now_; }
#else
#define RPROF(i)
#endif

// Persistent CTAs; cluster = the M = K*L mode frames of one view (cluster rank m = mode index),
// cluster c processes views c, c + n_clusters, ...  MT = compile-time M (0: run-time M).
template <int MT>
__global__ void __launch_bounds__(RNT, 1) regfft128_kernel(const RegArgs a)
{
    namespace cg = cooperative_groups;
    extern __shared__ __align__(16) unsigned char smem[];
    unsigned char *pbuf = smem;
    unsigned char *xbuf = smem + PBUF_BYTES;
    float2 *s_wy = reinterpret_cast<float2 *>(smem + PBUF_BYTES + XBUF3_BYTES);
    float2 *s_wx = s_wy + 128;
    __shared__ float red[4 * 32];
    __shared__ int s_rdcnt;                                     // warps that have finished reading the prefetch buffer in S1
    __shared__ uint32_t s_tmem;
    __shared__ __align__(8) uint64_t mb_lo, mb_hi, mb_amp;      // psi rows 0..63 (half A), rows 64..127 (half B), sqrt(I) (half A)

    const int tid = threadIdx.x, w = tid >> 5, t = tid & 31;
    const int M = MT ? MT : a.K * a.L;
    const int m = blockIdx.x % M, cl = blockIdx.x / M, ncl = gridDim.x / M;
    const int k = m / a.L, l = m % a.L;
    if (tid < 128) s_wy[tid] = a.wy[tid];
    else if (tid < 256) s_wx[tid - 128] = a.wx[tid - 128];
    if (tid == 0) {
        s_rdcnt = 0;
        mbar_init(&mb_lo, 1);
        mbar_init(&mb_hi, 1);
        mbar_init(&mb_amp, 1);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    if (w == 0) {       // all 512 TMEM columns (this kernel is the only resident CTA of its SM)
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n"
                     :: "r"((uint32_t)__cvta_generic_to_shared(&s_tmem)), "r"(512) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
    // this thread's private columns: lane quarter w % 4, column block (w / 4) * 128; psi_old | P*O
    const uint32_t t_psi = s_tmem + ((uint32_t)(32 * (w & 3)) << 16) + (uint32_t)(w >> 2) * 128u;
    const uint32_t t_po = t_psi + 64u;

    unsigned char *wbuf = xbuf + w * 4096, *wspare = xbuf + X1S_SPARE_OFF + w * X1S_SPARE;
    float2 *xb2 = reinterpret_cast<float2 *>(xbuf);
    const float2 *Pk = a.P + (size_t)k * RNN + w * RN + t;
    const float cfac = a.beta > 0.f ? 1.f / (float)RNN : 0.f;
    float e0 = 0.f, e1 = 0.f, e2 = 0.f, e3 = 0.f;
    int par = 0;
    if (tid == 0 && cl < a.n_views) {       // first frame: both halves now
        const unsigned char *src = reinterpret_cast<const unsigned char *>(a.psi + ((size_t)cl * M + m) * RNN);
        bulk_load(pbuf, src, 65536, &mb_lo);
        bulk_load(pbuf + 65536, src + 65536, 65536, &mb_hi);
    }

#ifdef DM_REG_PROF
    long long prof[8] = {0, 0, 0, 0, 0, 0, 0, 0}, tprev = clock64();
#endif
    int it = 0;
    for (int view = cl; view < a.n_views; view += ncl, par ^= 1, ++it) {
        const int2 p0 = a.pos[view];
        float2 *psi_f = a.psi + ((size_t)view * M + m) * RNN + w * RN + t;
        const float2 *Ow = a.O + (size_t)l * a.H * a.W + (size_t)(p0.x + w) * a.W + p0.y + t;
        const int nview = view + ncl;
        const unsigned char *nsrc = reinterpret_cast<const unsigned char *>(a.psi + ((size_t)nview * M + m) * RNN);
        float2 u[32];
        // ---- S1 + S2: R = 2 P O - psi in L0; psi_old and P*O parked in tensor memory ----
        // P and O come from L2: all of P and half of O are requested before anything else (psi still
        // sits in shared memory, so the registers are free), the other half of O while the first is used.
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
                    for (int r = 0; r < 4; ++r) u[4 * i + r] = ps[i * 16 * RN + r * 32];
                    tmem_st8(t_psi + 8 * i, u[4 * i], u[4 * i + 1], u[4 * i + 2], u[4 * i + 3]);
                    tmem_st8(t_po + 8 * i, po[4 * i], po[4 * i + 1], po[4 * i + 2], po[4 * i + 3]);
#pragma unroll
                    for (int r = 0; r < 4; ++r)
                        u[4 * i + r] = make_float2(2.f * po[4 * i + r].x - u[4 * i + r].x, 2.f * po[4 * i + r].y - u[4 * i + r].y);
                }
            }
        }
        // the warp that finishes reading the prefetch buffer LAST refills it; nobody waits (a block barrier here would
        // hold the warps whose P and O arrived early back from their first FFT pass)
        // release / acquire around the counter: the other warps' reads of pbuf are ordered before the refill by the
        // memory model (fence + atomic on both sides), not only by the data dependence of their tcgen05.st on the loads
        __syncwarp();
        if (t == 0) __threadfence_block();
        if (t == 0 && atomicAdd(&s_rdcnt, 1) == 15) {
            __threadfence_block();
            s_rdcnt = 0;
            asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
            bulk_load(pbuf, a.amp + (size_t)view * RNN, 65536, &mb_amp);
            if (nview < a.n_views) bulk_load(pbuf + 65536, nsrc + 65536, 65536, &mb_hi);
        }
        RPROF(0)
        tmem_wait_st();
        // ---- S3: forward 2-D FFT ----
        {
            float2 wy[8], wx[4];
#pragma unroll
            for (int q = 0; q < 8; ++q) wy[q] = s_wy[w * 8 + q];
#pragma unroll
            for (int r = 0; r < 4; ++r) wx[r] = s_wx[t * 4 + r];
            pass1_fwd(u, wy, wx);
        }
#pragma unroll
        for (int rho = 0; rho < 2; ++rho) {
            x1s_write(u, rho, t, wbuf, wspare);
            __syncwarp();
            x1s_read(u, rho, t, wbuf, wspare);
            __syncwarp();
        }
        pass2<false>(u);
        // exchange 2 in two rounds; M <= 2: the first half of pass 3 runs while the stores of the second round drain
        // (c1 -2 %; with the larger S4 code of M >= 3 the reordering costs spills: c2 +1.3 %, so not there)
        constexpr bool SPLIT3 = (MT == 1 || MT == 2);
        if (SPLIT3) {
            __syncthreads();
            x2_write(u, 0, w, t, xb2);
            __syncthreads();
            x2_read(u, 0, w, t, xb2);
            __syncthreads();
            x2_write(u, 1, w, t, xb2);
            pass3_half<false>(u, 0);
            __syncthreads();
            x2_read(u, 1, w, t, xb2);
            pass3_half<false>(u, 1);
        } else {
#pragma unroll
            for (int z = 0; z < 2; ++z) {
                __syncthreads();
                x2_write(u, z, w, t, xb2);
                __syncthreads();
                x2_read(u, z, w, t, xb2);
            }
            pass3<false>(u);
        }
        RPROF(1)
        // ---- S4: mode-summed modulus constraint (|F|^2 exchanged through L2) ----
        {
            float4 *mine = a.sbuf + (((size_t)par * gridDim.x + blockIdx.x) * 8) * RNT + tid;
            if (M > 1) {
#pragma unroll
                for (int j = 0; j < 8; ++j)
                    mine[j * RNT] = make_float4(abs2_rn(u[4 * j]), abs2_rn(u[4 * j + 1]), abs2_rn(u[4 * j + 2]), abs2_rn(u[4 * j + 3]));
                if (a.gbar) {
                    // the M CTAs of the view are not a hardware cluster (a cluster of M would leave SMs
                    // idle): release / acquire on a counter in L2; every CTA of the grid is resident
                    __syncthreads();
                    if (tid == 0) {
                        __threadfence();
                        atomicAdd(a.gbar + cl, 1);
                        const int want = M * (it + 1);
                        int v;
                        do {
                            asm volatile("ld.acquire.gpu.global.s32 %0, [%1];\n" : "=r"(v) : "l"(a.gbar + cl) : "memory");
                        } while (v < want);
                    }
                    __syncthreads();
                } else {
                    cluster_arrive();
                    cluster_wait();
                }
            } else {
                __syncthreads();
            }
            RPROF(2)
            mbar_wait(&mb_amp, par);
            const float4 *ampv = reinterpret_cast<const float4 *>(pbuf) + tid;
            const float4 *peers = a.sbuf + (((size_t)par * gridDim.x + (size_t)cl * M) * 8) * RNT + tid;
            // peers' |F|^2 come from L2: JB registers-quads per peer are requested at once
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
                    const float4 am = ampv[j * RNT];
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
                    for (int c = 0; c < 4; ++c) {
                        const float rs = rsqrtf(Sv[c] + a.eps);
                        const float d = Sv[c] * rs - av[c];
                        e0 = fmaf(d, d, e0);
                        e1 = fmaf(av[c], av[c], e1);
                        const float sc = av[c] * rs * cfac;
                        u[4 * j + c].x *= sc;
                        u[4 * j + c].y *= sc;
                    }
                }
            }
        }
        RPROF(3)
        // ---- S5: inverse 2-D FFT (mirror) ----
        if (SPLIT3) {
            pass3_half<true>(u, 0);
            __syncthreads();
            // every thread is past S4: half A (sqrt(I)) is free for the next frame's rows 0..63
            if (tid == 0 && nview < a.n_views) bulk_load(pbuf, nsrc, 65536, &mb_lo);
            x2_write(u, 0, w, t, xb2);
            pass3_half<true>(u, 1);             // while the stores of round 0 drain
            __syncthreads();
            x2_read(u, 0, w, t, xb2);
            __syncthreads();
            x2_write(u, 1, w, t, xb2);
            __syncthreads();
            x2_read(u, 1, w, t, xb2);
        } else {
            pass3<true>(u);
#pragma unroll
            for (int z = 0; z < 2; ++z) {
                __syncthreads();
                if (z == 0 && tid == 0 && nview < a.n_views) bulk_load(pbuf, nsrc, 65536, &mb_lo);
                x2_write(u, z, w, t, xb2);
                __syncthreads();
                x2_read(u, z, w, t, xb2);
            }
        }
        pass2<true>(u);
        // no block barrier: exchange 1 only touches what this warp itself read in exchange 2 and its spare strip
        __syncwarp();           // every lane's exchange-2 reads of that region are done before any lane overwrites it
#pragma unroll
        for (int rho = 0; rho < 2; ++rho) {
            x1s_write(u, rho, t, wbuf, wspare);
            __syncwarp();
            x1s_read(u, rho, t, wbuf, wspare);
            __syncwarp();
        }
        {
            float2 wy[8], wx[4];
#pragma unroll
            for (int q = 0; q < 8; ++q) wy[q] = s_wy[w * 8 + q];
#pragma unroll
            for (int r = 0; r < 4; ++r) wx[r] = s_wx[t * 4 + r];
            pass1_inv(u, wy, wx);
        }
        RPROF(4)
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
        RPROF(5)
    }
#ifdef DM_REG_PROF
    if (tid == 0 && it > 0 && (blockIdx.x == 0 || blockIdx.x == 1 || blockIdx.x == 100))
        printf("regfft128 blk %d, %d frames: S1+S2 %lld | forward FFT %lld | S4 store + group barrier %lld | S4 peers + scaling %lld | inverse FFT %lld | S6 %lld cycles per frame\n",
               blockIdx.x, it, prof[0] / it, prof[1] / it, prof[2] / it, prof[3] / it, prof[4] / it, prof[5] / it);
#endif
    asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
    __syncthreads();
    if (w == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" :: "r"(s_tmem), "r"(512) : "memory");
    float acc[4] = {m == 0 ? e0 : 0.f, m == 0 ? e1 : 0.f, e2 * a.beta * a.beta, e3};
    // deterministic block sum (xor tree in each warp, warps in order)
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int s = 16; s > 0; s >>= 1) acc[i] += __shfl_xor_sync(0xffffffffu, acc[i], s);
    if (t == 0)
#pragma unroll
        for (int i = 0; i < 4; ++i) red[i * 32 + w] = acc[i];
    __syncthreads();
    if (tid < 4) {
        float s = 0.f;
        for (int ww = 0; ww < 16; ++ww) s += red[tid * 32 + ww];
        a.part[(size_t)blockIdx.x * 4 + tid] = s;
    }
}

} // namespace dmreg
#endif // __CUDACC__
