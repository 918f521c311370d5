// dm_fft.cuh -- in-register radix butterflies and in-place tile passes of the 2-D FFT used by
// every psi-update kernel (steps S3/S5 of DESIGN.md; the F and F^-1 of eq. (3)).
//
// Scheme: decimation-in-frequency forward passes that leave the spectrum in DIGIT-REVERSED
// order along each axis, and mirrored decimation-in-time inverse passes that take exactly
// that order back to natural order.  The Fourier-modulus step (eq. (4)) is
// pointwise in q, so it runs on the permuted spectrum; sqrt(I) is stored once in the same
// permuted order (dm_set_data).  No bit-reversal pass is ever executed.
//
// Every function is __host__ __device__ so the CPU test-suite can run the very same pass
// code through dm_host_fft2 (include/dm.h) before anything goes to a GPU.
#pragma once
#include <cuda_runtime.h>

#define DM_HD __host__ __device__ __forceinline__

namespace dmfft {

// On the device complex add / subtract are ONE packed instruction each (Blackwell add.f32x2 /
// fma.rn.f32x2 with a -1 multiplier: same round-to-nearest results as two scalar adds, half the
// issue slots; the FP32 pipe still retires 128 lanes per clock).
#if defined(__CUDA_ARCH__) && __CUDA_ARCH__ >= 1000 && !defined(DM_NO_F32X2)
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return __ffma2_rn(b, make_float2(-1.f, -1.f), a); }
#else
DM_HD float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
DM_HD float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
#endif
DM_HD float2 cmul(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
// a * conj(b)
DM_HD float2 cmulc(float2 a, float2 b) { return make_float2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y); }
// multiply by -i (forward) or +i (inverse)
template <bool INV> DM_HD float2 mul_mi(float2 a) { return INV ? make_float2(-a.y, a.x) : make_float2(a.y, -a.x); }
DM_HD float cabs2(float2 a) { return a.x * a.x + a.y * a.y; }

// radices per axis for each supported frame edge (product = N); R3 = 1 when unused.
template <int N> struct Radix;
template <> struct Radix<64>  { static constexpr int R1 = 8,  R2 = 8,  R3 = 1; };
template <> struct Radix<128> { static constexpr int R1 = 8,  R2 = 16, R3 = 1; };
template <> struct Radix<256> { static constexpr int R1 = 16, R2 = 16, R3 = 1; };
template <> struct Radix<512> { static constexpr int R1 = 8,  R2 = 8,  R3 = 8; };

// ---- natural-order DFT_R of R values held in registers (forward: exp(-2 pi i nk/R)) ----
template <bool INV> DM_HD void dft2(float2 &a, float2 &b)
{
    float2 t = a;
    a = cadd(t, b);
    b = csub(t, b);
}

template <bool INV> DM_HD void dft4(float2 &a0, float2 &a1, float2 &a2, float2 &a3)
{
    float2 t0 = cadd(a0, a2), t1 = csub(a0, a2), t2 = cadd(a1, a3), t3 = mul_mi<INV>(csub(a1, a3));
    a0 = cadd(t0, t2);
    a2 = csub(t0, t2);
    a1 = cadd(t1, t3);
    a3 = csub(t1, t3);
}

template <bool INV> DM_HD void dft8(float2 (&u)[8])
{
    constexpr float H = 0.70710678118654752440f;
    // even / odd 4-point transforms (decimation in time)
    dft4<INV>(u[0], u[2], u[4], u[6]);   // E[0..3] in u[0],u[2],u[4],u[6]
    dft4<INV>(u[1], u[3], u[5], u[7]);   // O[0..3] in u[1],u[3],u[5],u[7]
    // O[k] *= w8^k
    float2 o1 = u[3], o2 = u[5], o3 = u[7];
    if (!INV) {
        o1 = make_float2((o1.x + o1.y) * H, (o1.y - o1.x) * H);      // (1 - i)/sqrt2
        o2 = make_float2(o2.y, -o2.x);                                // -i
        o3 = make_float2((o3.y - o3.x) * H, -(o3.x + o3.y) * H);     // (-1 - i)/sqrt2
    } else {
        o1 = make_float2((o1.x - o1.y) * H, (o1.x + o1.y) * H);      // (1 + i)/sqrt2
        o2 = make_float2(-o2.y, o2.x);                                // +i
        o3 = make_float2(-(o3.x + o3.y) * H, (o3.x - o3.y) * H);     // (-1 + i)/sqrt2
    }
    float2 e0 = u[0], e1 = u[2], e2 = u[4], e3 = u[6], o0 = u[1];
    u[0] = cadd(e0, o0); u[4] = csub(e0, o0);
    u[1] = cadd(e1, o1); u[5] = csub(e1, o1);
    u[2] = cadd(e2, o2); u[6] = csub(e2, o2);
    u[3] = cadd(e3, o3); u[7] = csub(e3, o3);
}

// w16^m = exp(-+ 2 pi i m / 16) for the m = n2*k1 that occur (n2,k1 in 1..3)
template <bool INV, int M> DM_HD float2 mul_w16(float2 a)
{
    constexpr float C1 = 0.92387953251128675613f, S1 = 0.38268343236508977173f;
    constexpr float H = 0.70710678118654752440f;
    constexpr float c = (M == 1) ? C1 : (M == 2) ? H : (M == 3) ? S1 : (M == 4) ? 0.f : (M == 6) ? -H : /*9*/ -C1;
    constexpr float s = (M == 1) ? S1 : (M == 2) ? H : (M == 3) ? C1 : (M == 4) ? 1.f : (M == 6) ? H : /*9*/ -S1;
    // forward: (c - i s); inverse: (c + i s)
    return INV ? make_float2(a.x * c - a.y * s, a.x * s + a.y * c)
               : make_float2(a.x * c + a.y * s, a.y * c - a.x * s);
}

template <bool INV> DM_HD void dft16(float2 (&u)[16])
{
    // n = 4 n1 + n2 ; A_n2[k1] = DFT4 over n1
    dft4<INV>(u[0], u[4], u[8],  u[12]);
    dft4<INV>(u[1], u[5], u[9],  u[13]);
    dft4<INV>(u[2], u[6], u[10], u[14]);
    dft4<INV>(u[3], u[7], u[11], u[15]);
    // A_n2[k1] lives in u[4 k1 + n2]; twiddle by w16^(n2 k1)
    u[5]  = mul_w16<INV, 1>(u[5]);  u[6]  = mul_w16<INV, 2>(u[6]);  u[7]  = mul_w16<INV, 3>(u[7]);
    u[9]  = mul_w16<INV, 2>(u[9]);  u[10] = mul_w16<INV, 4>(u[10]); u[11] = mul_w16<INV, 6>(u[11]);
    u[13] = mul_w16<INV, 3>(u[13]); u[14] = mul_w16<INV, 6>(u[14]); u[15] = mul_w16<INV, 9>(u[15]);
    // X[k1 + 4 k2] = DFT4 over n2 of u[4 k1 + n2]  -> result k2 lands in u[4 k1 + k2]
    dft4<INV>(u[0],  u[1],  u[2],  u[3]);
    dft4<INV>(u[4],  u[5],  u[6],  u[7]);
    dft4<INV>(u[8],  u[9],  u[10], u[11]);
    dft4<INV>(u[12], u[13], u[14], u[15]);
    // u[4 k1 + k2] holds X[k1 + 4 k2]: transpose the 4x4 register block to natural order
    float2 t;
    t = u[1];  u[1]  = u[4];  u[4]  = t;
    t = u[2];  u[2]  = u[8];  u[8]  = t;
    t = u[3];  u[3]  = u[12]; u[12] = t;
    t = u[6];  u[6]  = u[9];  u[9]  = t;
    t = u[7];  u[7]  = u[13]; u[13] = t;
    t = u[11]; u[11] = u[14]; u[14] = t;
}

template <int R, bool INV> struct Dft;
template <bool INV> struct Dft<2, INV>  { static DM_HD void run(float2 (&u)[2])  { dft2<INV>(u[0], u[1]); } };
template <bool INV> struct Dft<4, INV>  { static DM_HD void run(float2 (&u)[4])  { dft4<INV>(u[0], u[1], u[2], u[3]); } };
template <bool INV> struct Dft<8, INV>  { static DM_HD void run(float2 (&u)[8])  { dft8<INV>(u); } };
template <bool INV> struct Dft<16, INV> { static DM_HD void run(float2 (&u)[16]) { dft16<INV>(u); } };

// ---- shared-memory tile addressing --------------------------------------------------
// A tile is a row-major array of complex64; element e (linear index) is stored at swz(e):
// the 16-byte chunk index is XORed with bits of the 128-byte group index, so that
//   - 16 consecutive elements (one 128-B group) are a permutation of the same group
//     (lanes along x: conflict-free 64-bit accesses), and
//   - a thread that walks R consecutive elements while its neighbours walk the next groups
//     (the stride-1 x pass) hits 8 different 16-B bank groups per quarter warp.
DM_HD int swz(int e)
{
    int c = e >> 1;
    c ^= (c >> 3) & 7;
    return (c << 1) | (e & 1);
}

// One in-place pass over a tile with x extent W (elements) and y extent H (rows).
//   ALONG_Y = false: transform along x, one line per row   (needs NFFT == W)
//   ALONG_Y = true : transform along y, one line per column (needs NFFT == H)
// BLK = current block size of the decimation (NFFT for the first forward pass), R = radix.
// Forward (DIF): u = x[b*BLK + o + r*T]; v = DFT_R(u); x[.. q ..] = v[q] * w_BLK^(q o).
// Inverse (DIT) mirrors it: u[q] = x[..] * conj(w_BLK^(q o)); v = IDFT_R(u) (unscaled).
// tw[n] = exp(-2 pi i n / NFFT), n < NFFT.
template <int NFFT, int R, int BLK, bool INV, bool ALONG_Y, int W, int H>
DM_HD void tile_pass(float2 *tile, const float2 *tw, int tid, int nthr)
{
    constexpr int T = BLK / R;
    constexpr int NB = NFFT / R;                    // butterflies per line
    constexpr int LINES = ALONG_Y ? W : H;
    constexpr int TOTAL = LINES * NB;
    for (int id = tid; id < TOTAL; id += nthr) {
        int line, g;
        if (ALONG_Y) { line = id % W; g = id / W; }
        else         { g = id % NB;   line = id / NB; }
        const int b = g / T, o = g % T;
        const int base = b * BLK + o;
        float2 u[R];
        int addr[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int i = base + r * T;
            addr[r] = swz(ALONG_Y ? i * W + line : line * W + i);
            u[r] = tile[addr[r]];
        }
        if (INV && T > 1) {
#pragma unroll
            for (int q = 1; q < R; ++q) u[q] = cmulc(u[q], tw[q * o * (NFFT / BLK)]);
        }
        Dft<R, INV>::run(u);
        if (!INV && T > 1) {
#pragma unroll
            for (int q = 1; q < R; ++q) u[q] = cmul(u[q], tw[q * o * (NFFT / BLK)]);
        }
#pragma unroll
        for (int r = 0; r < R; ++r) tile[addr[r]] = u[r];
    }
}

// All passes of one axis.  SYNC is a functor called between passes (block barrier on the
// device, nothing on the host emulation).
template <int N, bool INV, bool ALONG_Y, int W, int H, class SYNC>
DM_HD void axis_fft(float2 *tile, const float2 *tw, int tid, int nthr, SYNC sync)
{
    using Rx = Radix<N>;
    constexpr int B1 = N, B2 = N / Rx::R1, B3 = N / (Rx::R1 * Rx::R2);
    if (!INV) {
        tile_pass<N, Rx::R1, B1, false, ALONG_Y, W, H>(tile, tw, tid, nthr);
        sync();
        tile_pass<N, Rx::R2, B2, false, ALONG_Y, W, H>(tile, tw, tid, nthr);
        sync();
        if (Rx::R3 > 1) {
            tile_pass<N, (Rx::R3 > 1 ? Rx::R3 : 2), (Rx::R3 > 1 ? B3 : 2), false, ALONG_Y, W, H>(tile, tw, tid, nthr);
            sync();
        }
    } else {
        if (Rx::R3 > 1) {
            tile_pass<N, (Rx::R3 > 1 ? Rx::R3 : 2), (Rx::R3 > 1 ? B3 : 2), true, ALONG_Y, W, H>(tile, tw, tid, nthr);
            sync();
        }
        tile_pass<N, Rx::R2, B2, true, ALONG_Y, W, H>(tile, tw, tid, nthr);
        sync();
        tile_pass<N, Rx::R1, B1, true, ALONG_Y, W, H>(tile, tw, tid, nthr);
        sync();
    }
}

// position p (after the forward passes) -> frequency index k it holds
template <int N> inline int digit_reverse(int p)
{
    using Rx = Radix<N>;
    const int T1 = N / Rx::R1, T2 = T1 / Rx::R2;
    const int q1 = p / T1, q2 = (p % T1) / T2, q3 = p % T2;     // T3 == 1
    return q1 + Rx::R1 * q2 + Rx::R1 * Rx::R2 * q3;
}

} // namespace dmfft
