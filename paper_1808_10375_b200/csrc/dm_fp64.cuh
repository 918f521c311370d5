// dm_fp64.cuh -- the whole DM iteration in DOUBLE precision (the paper's own precision,
// PAPER.md:130 "all of the calculations are done in double precision"), as a validation mode
// (DM_PARAM_PRECISION = 1).  Plain kernels, no tuning: its purpose is the
// long free-running parity against the FP64 oracle, which FP32 arithmetic cannot show because
// the DM transient amplifies rounding differences.
//
//   psi update (eqs. (2)-(4)):  rows64 (R = 2PO - psi, FFT_x) -> cols64 (FFT_y) -> modulus64
//                               -> cols64 (IFFT_y) -> rows64 (IFFT_x, psi += beta (G - PO))
//   object / probe update (eqs. (6), (5)):  object64 (coverage lists, j then k ascending),
//                               probe64 (j then l ascending) -- the definition's summation orders
//   errors (eq. (7)):           per-CTA partial pairs, err64_finalize (fixed order)
// One CTA transforms one line of N points in shared memory: textbook radix-2 decimation in time.
#pragma once
#include <cuda_runtime.h>

namespace dm64 {

typedef double2 cd;

__device__ __forceinline__ cd cmul(cd a, cd b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ double cabs2(cd a) { return a.x * a.x + a.y * a.y; }

struct Args {
    int N, logN, n_views, K, L, H, W;
    const int2 *pos;
    const cd *P, *O;            // [K][N][N], [L][H][W]
    cd *psi;                    // [n_views][M][N][N]
    cd *scratch;                // [n_views][M][N][N] spectra
    const double *amp;          // [n_views][N][N] sqrt(I), natural order
    const cd *tw;               // [N/2] exp(-2 pi i n / N)
    double beta, eps;
    double *partF, *partS;      // [n_views * N / 256 ...][2], [MV * N][2]
};

// in-place FFT of the N values in `s` (shared), N/2 threads; forward: exp(-i...), inverse: conjugate, unscaled
template <bool INV> __device__ void line_fft(cd *s, const cd *tw, int N, int logN)
{
    const int t = threadIdx.x;
    for (int st = 0; st < logN; ++st) {
        const int half = 1 << st;
        const int j = t & (half - 1), base = ((t >> st) << (st + 1)) + j;
        cd w = tw[j * (N >> (st + 1))];
        if (INV) w.y = -w.y;
        __syncthreads();
        const cd a = s[base], b = cmul(s[base + half], w);
        s[base] = make_double2(a.x + b.x, a.y + b.y);
        s[base + half] = make_double2(a.x - b.x, a.y - b.y);
    }
    __syncthreads();
}

__device__ __forceinline__ int bitrev(int x, int logN) { return (int)(__brev((unsigned)x) >> (32 - logN)); }

// deterministic CTA sum of two doubles per thread -> thread 0 (binary tree over a power-of-two block)
__device__ __forceinline__ void cta_sum2(double &a, double &b, double *sh)
{
    const int n = blockDim.x;
    sh[threadIdx.x] = a;
    sh[n + threadIdx.x] = b;
    __syncthreads();
    for (int w = n >> 1; w > 0; w >>= 1) {
        if ((int)threadIdx.x < w) {
            sh[threadIdx.x] += sh[threadIdx.x + w];
            sh[n + threadIdx.x] += sh[n + threadIdx.x + w];
        }
        __syncthreads();
    }
    a = sh[0];
    b = sh[n];
}

// one CTA = row y of mode frame f.  FWD: R = 2 P O - psi, FFT along x -> scratch.
// !FWD: IFFT along x of scratch (1/N^2 applied), psi += beta (G - P O), error partials.
template <bool FWD> __global__ void rows64_kernel(const Args a)
{
    extern __shared__ double2 sm64[];
    cd *s = sm64;
    double *sh = reinterpret_cast<double *>(sm64 + a.N);
    const int N = a.N, M = a.K * a.L;
    const size_t NN = (size_t)N * N;
    const int f = blockIdx.x / N, y = blockIdx.x % N;
    const int view = f / M, m = f % M, k = m / a.L, l = m % a.L;
    const int2 p0 = a.pos[view];
    const cd *Prow = a.P + (size_t)k * NN + (size_t)y * N;
    const cd *Orow = a.O + (size_t)l * a.H * a.W + (size_t)(p0.x + y) * a.W + p0.y;
    cd *psi = a.psi + (size_t)f * NN + (size_t)y * N;
    cd *scr = a.scratch + (size_t)f * NN + (size_t)y * N;
    if (FWD) {
        for (int x = threadIdx.x; x < N; x += blockDim.x) {
            const cd po = cmul(Prow[x], Orow[x]), ps = psi[x];
            s[bitrev(x, a.logN)] = make_double2(2.0 * po.x - ps.x, 2.0 * po.y - ps.y);
        }
        line_fft<false>(s, a.tw, N, a.logN);
        for (int x = threadIdx.x; x < N; x += blockDim.x) scr[x] = s[x];
    } else {
        for (int x = threadIdx.x; x < N; x += blockDim.x) s[bitrev(x, a.logN)] = scr[x];
        line_fft<true>(s, a.tw, N, a.logN);
        const double inv = 1.0 / ((double)N * (double)N);
        double e0 = 0.0, e1 = 0.0;
        for (int x = threadIdx.x; x < N; x += blockDim.x) {
            const cd po = cmul(Prow[x], Orow[x]), ps = psi[x];
            const double dx = a.beta * (s[x].x * inv - po.x), dy = a.beta * (s[x].y * inv - po.y);
            const cd nw = make_double2(ps.x + dx, ps.y + dy);
            e0 += dx * dx + dy * dy;
            e1 += nw.x * nw.x + nw.y * nw.y;
            psi[x] = nw;
        }
        cta_sum2(e0, e1, sh);
        if (threadIdx.x == 0) {
            a.partS[2 * (size_t)blockIdx.x] = e0;
            a.partS[2 * (size_t)blockIdx.x + 1] = e1;
        }
    }
}

// one CTA = column x of mode frame f, in place in scratch
template <bool INV> __global__ void cols64_kernel(const Args a)
{
    extern __shared__ double2 sm64[];
    cd *s = sm64;
    const int N = a.N;
    const size_t NN = (size_t)N * N;
    const int f = blockIdx.x / N, x = blockIdx.x % N;
    cd *col = a.scratch + (size_t)f * NN + x;
    for (int y = threadIdx.x; y < N; y += blockDim.x) s[bitrev(y, a.logN)] = col[(size_t)y * N];
    line_fft<INV>(s, a.tw, N, a.logN);
    for (int y = threadIdx.x; y < N; y += blockDim.x) col[(size_t)y * N] = s[y];
}

// eq. (4): S = sum over modes |F|^2, scale = amp / sqrt(S + eps); grid = (NN / 256, n_views), 256 threads
__global__ void modulus64_kernel(const Args a)
{
    __shared__ double sh[512];
    const int N = a.N, M = a.K * a.L;
    const size_t NN = (size_t)N * N;
    const int view = blockIdx.y;
    const size_t q = (size_t)blockIdx.x * 256 + threadIdx.x;
    cd *F = a.scratch + (size_t)view * M * NN + q;
    double S = 0.0;
    for (int m = 0; m < M; ++m) S += cabs2(F[(size_t)m * NN]);
    const double amp = a.amp[(size_t)view * NN + q];
    const double d = sqrt(S) - amp;
    double e0 = d * d, e1 = amp * amp;
    const double sc = amp / sqrt(S + a.eps);
    for (int m = 0; m < M; ++m) {
        cd v = F[(size_t)m * NN];
        F[(size_t)m * NN] = make_double2(v.x * sc, v.y * sc);
    }
    cta_sum2(e0, e1, sh);
    if (threadIdx.x == 0) {
        const size_t o = (size_t)view * gridDim.x + blockIdx.x;
        a.partF[2 * o] = e0;
        a.partF[2 * o + 1] = e1;
    }
}

// eq. (6): one thread per object pixel, one CTA per OBJ_TH x OBJ_TW tile (the FP32 path's coverage
// lists); j ascending, k ascending inside = the definition's order.  part: [tiles][L][2]
__global__ void object64_kernel(int N, int K, int L, int H, int W, int TH, int TW, const int2 *__restrict__ pos,
                                const int *__restrict__ tile_ptr, const int *__restrict__ tile_views,
                                const cd *__restrict__ P, const cd *__restrict__ psi, const cd *__restrict__ O_old,
                                cd *__restrict__ O_new, const double *__restrict__ alphas, double *__restrict__ part,
                                double *__restrict__ den_out)
{
    __shared__ double sh[512];
    const size_t NN = (size_t)N * N, HW = (size_t)H * W;
    const int ntx = (W + TW - 1) / TW;
    const int tile = blockIdx.x, ty = tile / ntx, tx = tile % ntx;
    const int y = ty * TH + threadIdx.x / TW, x = tx * TW + threadIdx.x % TW;
    const bool inb = y < H && x < W;
    const int beg = tile_ptr[tile], end = tile_ptr[tile + 1];
    const double alpha = alphas[0];
    for (int l = 0; l < L; ++l) {
        double nx = 0.0, ny = 0.0, den = 0.0;
        if (inb)
            for (int i = beg; i < end; ++i) {
                const int j = tile_views[i];
                const int2 p0 = pos[j];
                const int ry = y - p0.x, rx = x - p0.y;
                if ((unsigned)ry < (unsigned)N && (unsigned)rx < (unsigned)N) {
                    const size_t r = (size_t)ry * N + rx;
                    for (int k = 0; k < K; ++k) {
                        const cd p = P[(size_t)k * NN + r];
                        const cd s = psi[((size_t)j * K * L + (size_t)k * L + l) * NN + r];
                        nx += p.x * s.x + p.y * s.y;
                        ny += p.x * s.y - p.y * s.x;
                        den += cabs2(p);
                    }
                }
            }
        double e0 = 0.0, e1 = 0.0;
        if (inb) {
            const size_t o = (size_t)l * HW + (size_t)y * W + x;
            const cd oo = O_old[o];
            cd on = oo;
            const double dd = alpha + den;
            if (dd > 0.0) on = make_double2((alpha * oo.x + nx) / dd, (alpha * oo.y + ny) / dd);
            O_new[o] = on;
            if (den_out && l == 0) den_out[(size_t)y * W + x] = den;
            e0 = (on.x - oo.x) * (on.x - oo.x) + (on.y - oo.y) * (on.y - oo.y);
            e1 = cabs2(on);
        }
        cta_sum2(e0, e1, sh);
        if (threadIdx.x == 0) {
            part[((size_t)tile * L + l) * 2] = e0;
            part[((size_t)tile * L + l) * 2 + 1] = e1;
        }
        __syncthreads();
    }
}

// eq. (5): one thread per probe pixel, blockIdx.y = probe mode k; j ascending, l ascending.  part: [blocks][K][2]
__global__ void probe64_kernel(int N, int K, int L, int n_views, int H, int W, const int2 *__restrict__ pos,
                               const cd *__restrict__ O, const cd *__restrict__ psi, const cd *__restrict__ P_old,
                               cd *__restrict__ P_new, const double *__restrict__ alphas, double *__restrict__ part,
                               double *__restrict__ den_out)
{
    __shared__ double sh[512];
    const size_t NN = (size_t)N * N, HW = (size_t)H * W;
    const int r = blockIdx.x * blockDim.x + threadIdx.x, k = blockIdx.y;
    const int ry = r / N, rx = r % N;
    double nx = 0.0, ny = 0.0, den = 0.0;
    for (int j = 0; j < n_views; ++j) {
        const int2 p0 = pos[j];
        const cd *ob = O + (size_t)(p0.x + ry) * W + p0.y + rx;
        for (int l = 0; l < L; ++l) {
            const cd o = ob[(size_t)l * HW];
            const cd s = psi[((size_t)j * K * L + (size_t)k * L + l) * NN + r];
            nx += o.x * s.x + o.y * s.y;
            ny += o.x * s.y - o.y * s.x;
            den += cabs2(o);
        }
    }
    const double alpha = alphas[1], dd = alpha + den;
    const cd po = P_old[(size_t)k * NN + r];
    cd pn = po;
    if (dd > 0.0) pn = make_double2((alpha * po.x + nx) / dd, (alpha * po.y + ny) / dd);
    P_new[(size_t)k * NN + r] = pn;
    if (den_out && k == 0) den_out[r] = den;
    double e0 = (pn.x - po.x) * (pn.x - po.x) + (pn.y - po.y) * (pn.y - po.y), e1 = cabs2(pn);
    cta_sum2(e0, e1, sh);
    if (threadIdx.x == 0) {
        part[((size_t)blockIdx.x * K + k) * 2] = e0;
        part[((size_t)blockIdx.x * K + k) * 2 + 1] = e1;
    }
}

// one CTA per column of the error row: value = sqrt(sum num / sum den), 0/0 := 0, fixed order
struct Err64 {
    const double *pF; int nF;      // pairs
    const double *pS; int nS;
    const double *pP; int nP;      // [nP][K][2]
    const double *pO; int nO;      // [nO][L][2]
    int K, L;
    double *row;
};
__global__ void err64_finalize_kernel(const Err64 a)
{
    __shared__ double sh[2048];
    const int q = blockIdx.x;
    const double *p; int n, s;
    if (q == 0) { p = a.pF; n = a.nF; s = 2; }
    else if (q == 1) { p = a.pS; n = a.nS; s = 2; }
    else if (q < 2 + a.K) { p = a.pP + 2 * (q - 2); n = a.nP; s = 2 * a.K; }
    else { p = a.pO + 2 * (q - 2 - a.K); n = a.nO; s = 2 * a.L; }
    double num = 0.0, den = 0.0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        num += p[(size_t)i * s];
        den += p[(size_t)i * s + 1];
    }
    cta_sum2(num, den, sh);
    if (threadIdx.x == 0) a.row[q] = den > 0.0 ? sqrt(num / den) : 0.0;
}

// ---- conversions, initial state, maxima ---------------------------------------------------
__global__ void f2d_kernel(const float *__restrict__ in, double *__restrict__ out, size_t n, int take_sqrt)
{
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        out[i] = take_sqrt ? sqrt((double)in[i]) : (double)in[i];
}
__global__ void d2f_kernel(const double *__restrict__ in, float *__restrict__ out, size_t n)
{
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) out[i] = (float)in[i];
}
__global__ void psi_init64_kernel(int N, int K, int L, int H, int W, const int2 *__restrict__ pos,
                                  const cd *__restrict__ P, const cd *__restrict__ O, cd *__restrict__ psi)
{
    const size_t NN = (size_t)N * N;
    const int M = K * L, f = blockIdx.y, j = f / M, m = f % M, k = m / L, l = m % L;
    const int2 p0 = pos[j];
    for (size_t r = blockIdx.x * (size_t)blockDim.x + threadIdx.x; r < NN; r += (size_t)gridDim.x * blockDim.x) {
        const int ry = (int)(r / N), rx = (int)(r % N);
        psi[(size_t)f * NN + r] = cmul(P[(size_t)k * NN + r], O[(size_t)l * H * W + (size_t)(p0.x + ry) * W + p0.y + rx]);
    }
}
__global__ void max_scale64_kernel(const double *__restrict__ x, size_t n, double factor, double *out)
{
    __shared__ double sh[1024];
    double m = 0.0;
    for (size_t i = threadIdx.x; i < n; i += blockDim.x) m = fmax(m, x[i]);
    sh[threadIdx.x] = m;
    __syncthreads();
    for (int w = blockDim.x >> 1; w > 0; w >>= 1) {
        if ((int)threadIdx.x < w) sh[threadIdx.x] = fmax(sh[threadIdx.x], sh[threadIdx.x + w]);
        __syncthreads();
    }
    if (threadIdx.x == 0) out[0] = factor * sh[0];
}

} // namespace dm64
