/*
 * dm_oracle.c -- TEST INFRASTRUCTURE ONLY.  NOT part of the product path.
 *
 * Plain, slow, obviously-correct CPU restatement of the multi-mode difference-map (DM)
 * iteration of arXiv:1808.10375 Section II, eqs. (1)-(7), in
 * double-precision complex, with its own textbook radix-2 FFT.  It shares no code,
 * header, table or constant generator with the CUDA path under
 * paper_1808_10375_b200/csrc/; only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may load it.
 *
 * Order of one iteration (readings A3/A4 of DESIGN.md):
 *   A. psi update for every view, eq. (3) with the constrained transform eq. (4)
 *   B. object update eq. (6)  (old P, new psi)
 *   C. probe  update eq. (5)  (new O, new psi)
 *   D. error row: eps_F, eps_psi, eps_P[k], eps_O[l]  (eq. (7) and DESIGN.md A10)
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): brute-force O(N^4) DFT on 8x8 / 16x16,
 * Parseval, delta/constant transforms, round trip, numpy.fft cross-check; modulus
 * projection idempotence and |F'|^2 sum == I; DM fixed point on noise-free data;
 * fused-form identity; overlap projection closed forms and least-squares property;
 * a dense-DFT-matrix numpy restatement of 3 whole iterations on a tiny case;
 * equivariances; tables against brute force; the view-range entry points at the end of
 * this file (streaming of configs 3, 4) bit-identical to the monolithic steps for any split
 * of the views and to oracle_iterate over two iterations.  Convergence magnitudes on config 0 are
 * reported only: "parity unpinned" versus any published number (the paper prints none).
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC (see oracle/build.py).  -DORACLE_REAL=float
 * builds the FP32 yardstick of DESIGN.md protocol P4 (never used as truth).
 *
 * Layouts (all host pointers, row-major, complex interleaved re,im):
 *   psi  [n_views][K][L][N][N]   P [K][N][N]   O [L][H][W]   I/amp [n_views][N][N]
 *   positions int32 [n_views][2] = (y0, x0): probe pixel (ry,rx) meets object pixel
 *   (y0+ry, x0+rx)  (reading A5).
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifndef ORACLE_REAL
#define ORACLE_REAL double
#endif
typedef ORACLE_REAL real;
typedef ORACLE_REAL _Complex cplx;

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

static inline real cabs2(cplx z) { return creal(z) * creal(z) + cimag(z) * cimag(z); }

/* ------------------------------------------------------------------ FFT ---- */
/* Textbook iterative radix-2 decimation-in-time FFT, in place, length n = 2^m.
 * Forward: X[u] = sum_x x[x] exp(-2 pi i u x / n), unnormalised (reading A6).
 * tw[k] = exp(-2 pi i k / n), k < n/2, computed in double.                       */
static void make_twiddles(int n, cplx *tw)
{
    for (int k = 0; k < n / 2; ++k) {
        double a = -2.0 * M_PI * (double)k / (double)n;
        tw[k] = (real)cos(a) + (real)sin(a) * I;
    }
}

static void fft1d(cplx *x, int n, const cplx *tw, int inverse)
{
    for (int i = 1, j = 0; i < n; ++i) {            /* bit reversal permutation */
        int bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) { cplx t = x[i]; x[i] = x[j]; x[j] = t; }
    }
    for (int len = 2; len <= n; len <<= 1) {
        int half = len >> 1, stride = n / len;
        for (int s = 0; s < n; s += len)
            for (int k = 0; k < half; ++k) {
                cplx w = tw[k * stride];
                if (inverse) w = conj(w);
                cplx a = x[s + k], b = w * x[s + k + half];
                x[s + k] = a + b;
                x[s + k + half] = a - b;
            }
    }
}

/* 2-D transform of an N x N frame: rows (x, axis 1) then columns (y, axis 0).
 * Inverse includes the 1/N^2 factor (numpy convention, reading A6).              */
static void fft2_inplace(cplx *a, int N, const cplx *tw, int inverse, cplx *col)
{
    for (int y = 0; y < N; ++y) fft1d(a + (size_t)y * N, N, tw, inverse);
    for (int x = 0; x < N; ++x) {
        for (int y = 0; y < N; ++y) col[y] = a[(size_t)y * N + x];
        fft1d(col, N, tw, inverse);
        for (int y = 0; y < N; ++y) a[(size_t)y * N + x] = col[y];
    }
    if (inverse) {
        real s = (real)1 / ((real)N * (real)N);
        for (size_t i = 0; i < (size_t)N * N; ++i) a[i] *= s;
    }
}

static int is_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }

/* public: out = FFT2(in) (inverse != 0: IFFT2).  Returns 0, or -1 if N is not 2^m. */
int oracle_fft2(int N, const real *in, real *out, int inverse)
{
    if (!is_pow2(N)) return -1;
    cplx *tw = malloc(sizeof(cplx) * (N / 2 + 1)), *col = malloc(sizeof(cplx) * N);
    make_twiddles(N, tw);
    memcpy(out, in, sizeof(cplx) * (size_t)N * N);
    fft2_inplace((cplx *)out, N, tw, inverse, col);
    free(tw); free(col);
    return 0;
}

/* ---------------------------------------------------- integer tables (S0) ---- */
/* window table: (y0, x0, y0*W + x0) per view (S0).                      */
void oracle_window_table(int n_views, const int32_t *positions, int obj_w, int32_t *out)
{
    for (int j = 0; j < n_views; ++j) {
        out[3 * j + 0] = positions[2 * j];
        out[3 * j + 1] = positions[2 * j + 1];
        out[3 * j + 2] = positions[2 * j] * obj_w + positions[2 * j + 1];
    }
}

/* coverage lists: for every tile (ty,tx) of tile_h x tile_w object pixels, row-major,
 * the ascending list of views whose N x N window intersects it.  tile_ptr has
 * n_tiles+1 entries.  Call with tile_views == NULL to get the count only.
 * Written view-by-tile on purpose (the definition), not by inverting ranges.       */
int64_t oracle_coverage(int N, int n_views, const int32_t *positions, int obj_h, int obj_w,
                        int tile_h, int tile_w, int32_t *tile_ptr, int32_t *tile_views)
{
    int nty = (obj_h + tile_h - 1) / tile_h, ntx = (obj_w + tile_w - 1) / tile_w;
    int64_t nnz = 0;
    for (int ty = 0; ty < nty; ++ty)
        for (int tx = 0; tx < ntx; ++tx) {
            int ya = ty * tile_h, yb = ya + tile_h, xa = tx * tile_w, xb = xa + tile_w;
            if (tile_ptr) tile_ptr[ty * ntx + tx] = (int32_t)nnz;
            for (int j = 0; j < n_views; ++j) {
                int y0 = positions[2 * j], x0 = positions[2 * j + 1];
                if (y0 < yb && y0 + N > ya && x0 < xb && x0 + N > xa) {
                    if (tile_views) tile_views[nnz] = j;
                    ++nnz;
                }
            }
        }
    if (tile_ptr) tile_ptr[nty * ntx] = (int32_t)nnz;
    return nnz;
}

/* per-pixel number of covering views, int32 [H][W]. */
void oracle_cover_count(int N, int n_views, const int32_t *positions, int obj_h, int obj_w,
                        int32_t *count)
{
    memset(count, 0, sizeof(int32_t) * (size_t)obj_h * obj_w);
    for (int j = 0; j < n_views; ++j)
        for (int ry = 0; ry < N; ++ry)
            for (int rx = 0; rx < N; ++rx)
                count[(size_t)(positions[2 * j] + ry) * obj_w + positions[2 * j + 1] + rx] += 1;
}

/* ------------------------------------------------------ stateless steps ---- */
/* Constrained transform eq. (4) on M = K*L spectra of one view:
 *   S(q) = sum_m |F_m(q)|^2 ; scale = amp/sqrt(S + eps) ; F'_m = scale * F_m.
 * Also returns sum_q (sqrt(S)-amp)^2 in *err_num (A10).                  */
void oracle_modulus_project(int N, int M, const real *F_in, const real *amp, real eps,
                            real *F_out, real *err_num)
{
    const cplx *F = (const cplx *)F_in;
    cplx *G = (cplx *)F_out;
    size_t NN = (size_t)N * N;
    real e = 0;
    for (size_t q = 0; q < NN; ++q) {
        real S = 0;
        for (int m = 0; m < M; ++m) S += cabs2(F[m * NN + q]);
        real d = sqrt(S) - amp[q];
        e += d * d;
        real scale = amp[q] / sqrt(S + eps);
        for (int m = 0; m < M; ++m) G[m * NN + q] = scale * F[m * NN + q];
    }
    if (err_num) *err_num = e;
}

/* Step A for ONE view, eq. (3):
 *   PO = P_k * O_l|window ; R = 2 PO - psi ; F = FFT2(R) ; F' = F_c ; G = IFFT2(F')
 *   psi <- psi + beta (G - PO).
 * psi is [K][L][N][N] in/out.  acc[0] += sum (sqrt(S)-amp)^2, acc[1] += sum amp^2,
 * acc[2] += sum |beta (G-PO)|^2, acc[3] += sum |psi_new|^2.
 * fused != 0 evaluates the algebraically equal form
 *   psi <- (2-beta) PO + IFFT2[(beta*scale - 1) F]          (DESIGN.md identity pin)   */
void oracle_view_update(int N, int K, int L, const real *P_in, const real *O_in, int obj_h,
                        int obj_w, int y0, int x0, real *psi_io, const real *amp, real beta,
                        real eps, real *acc, int fused)
{
    (void)obj_h;
    const cplx *P = (const cplx *)P_in, *O = (const cplx *)O_in;
    cplx *psi = (cplx *)psi_io;
    size_t NN = (size_t)N * N;
    int M = K * L;
    cplx *PO = malloc(sizeof(cplx) * NN * M), *F = malloc(sizeof(cplx) * NN * M);
    cplx *tw = malloc(sizeof(cplx) * (N / 2 + 1)), *col = malloc(sizeof(cplx) * N);
    make_twiddles(N, tw);
    for (int k = 0; k < K; ++k)
        for (int l = 0; l < L; ++l) {
            int m = k * L + l;
            for (int ry = 0; ry < N; ++ry)
                for (int rx = 0; rx < N; ++rx) {
                    size_t r = (size_t)ry * N + rx;
                    cplx po = P[k * NN + r] *
                              O[(size_t)l * obj_h * obj_w + (size_t)(y0 + ry) * obj_w + x0 + rx];
                    PO[m * NN + r] = po;
                    F[m * NN + r] = 2 * po - psi[m * NN + r];
                }
            fft2_inplace(F + m * NN, N, tw, 0, col);
        }
    for (size_t q = 0; q < NN; ++q) {
        real S = 0;
        for (int m = 0; m < M; ++m) S += cabs2(F[m * NN + q]);
        real d = sqrt(S) - amp[q];
        acc[0] += d * d;
        acc[1] += amp[q] * amp[q];
        real scale = amp[q] / sqrt(S + eps);
        for (int m = 0; m < M; ++m)
            F[m * NN + q] *= fused ? (beta * scale - 1) : scale;
    }
    for (int m = 0; m < M; ++m) {
        fft2_inplace(F + m * NN, N, tw, 1, col);
        for (size_t r = 0; r < NN; ++r) {
            cplx old = psi[m * NN + r], nw;
            if (fused) nw = (2 - beta) * PO[m * NN + r] + F[m * NN + r];
            else       nw = old + beta * (F[m * NN + r] - PO[m * NN + r]);
            acc[2] += cabs2(nw - old);
            acc[3] += cabs2(nw);
            psi[m * NN + r] = nw;
        }
    }
    free(PO); free(F); free(tw); free(col);
}

/* Step B, eq. (6): for every l and object pixel, j ascending, k ascending.
 *   O_new = (alpha*O + num)/(alpha + den) if alpha+den > 0 else O   (reading A8; alpha = 0
 *   is the paper's literal quotient).  den is shared by all l (reading A15).            */
void oracle_object_update(int N, int n_views, int K, int L, int obj_h, int obj_w,
                          const int32_t *positions, const real *P_in, const real *psi_in,
                          const real *O_old_in, real alpha, real *O_new_out)
{
    const cplx *P = (const cplx *)P_in, *psi = (const cplx *)psi_in, *Oo = (const cplx *)O_old_in;
    cplx *On = (cplx *)O_new_out;
    size_t NN = (size_t)N * N, HW = (size_t)obj_h * obj_w;
#pragma omp parallel for schedule(static)
    for (int y = 0; y < obj_h; ++y)
        for (int x = 0; x < obj_w; ++x)
            for (int l = 0; l < L; ++l) {
                cplx num = 0; real den = 0;
                for (int j = 0; j < n_views; ++j) {
                    int ry = y - positions[2 * j], rx = x - positions[2 * j + 1];
                    if (ry < 0 || ry >= N || rx < 0 || rx >= N) continue;
                    size_t r = (size_t)ry * N + rx;
                    for (int k = 0; k < K; ++k) {
                        cplx p = P[k * NN + r];
                        num += conj(p) * psi[(((size_t)j * K + k) * L + l) * NN + r];
                        den += cabs2(p);
                    }
                }
                size_t o = l * HW + (size_t)y * obj_w + x;
                On[o] = (alpha + den > 0) ? (alpha * Oo[o] + num) / (alpha + den) : Oo[o];
            }
}

/* Step C, eq. (5): for every k and probe pixel, j ascending, l ascending. */
void oracle_probe_update(int N, int n_views, int K, int L, int obj_h, int obj_w,
                         const int32_t *positions, const real *O_in, const real *psi_in,
                         const real *P_old_in, real alpha, real *P_new_out)
{
    const cplx *O = (const cplx *)O_in, *psi = (const cplx *)psi_in, *Po = (const cplx *)P_old_in;
    cplx *Pn = (cplx *)P_new_out;
    size_t NN = (size_t)N * N, HW = (size_t)obj_h * obj_w;
#pragma omp parallel for schedule(static)
    for (int ry = 0; ry < N; ++ry)
        for (int rx = 0; rx < N; ++rx)
            for (int k = 0; k < K; ++k) {
                size_t r = (size_t)ry * N + rx;
                cplx num = 0; real den = 0;
                for (int j = 0; j < n_views; ++j)
                    for (int l = 0; l < L; ++l) {
                        cplx o = O[l * HW + (size_t)(positions[2 * j] + ry) * obj_w +
                                   positions[2 * j + 1] + rx];
                        num += conj(o) * psi[(((size_t)j * K + k) * L + l) * NN + r];
                        den += cabs2(o);
                    }
                Pn[k * NN + r] = (alpha + den > 0) ? (alpha * Po[k * NN + r] + num) / (alpha + den)
                                                    : Po[k * NN + r];
            }
}

/* eq. (7): sqrt( sum|new-old|^2 / sum|new|^2 ), 0/0 := 0. */
real oracle_rel_change(size_t n, const real *new_in, const real *old_in)
{
    const cplx *a = (const cplx *)new_in, *b = (const cplx *)old_in;
    real num = 0, den = 0;
    for (size_t i = 0; i < n; ++i) { num += cabs2(a[i] - b[i]); den += cabs2(a[i]); }
    return den > 0 ? sqrt(num / den) : 0;
}

/* ------------------------------------------------------------ stateful ---- */
typedef struct oracle_dm {
    int N, n_views, K, L, H, W;
    int32_t *pos;
    real beta, a_obj, a_probe, eps_f;       /* a_* are RELATIVE factors (reading A8) */
    real alpha_obj, alpha_probe;            /* absolute, frozen at set_data            */
    cplx *P, *O, *psi;
    real *amp;
    int has_data, n_rows, cap_rows;
    double *errors;                          /* [rows][2+K+L] */
} oracle_dm;

oracle_dm *oracle_create(int N, int n_views, int K, int L, int obj_h, int obj_w,
                         const int32_t *positions)
{
    if (!is_pow2(N) || n_views <= 0 || K <= 0 || L <= 0 || !positions) return NULL;
    for (int j = 0; j < n_views; ++j)
        if (positions[2 * j] < 0 || positions[2 * j] + N > obj_h || positions[2 * j + 1] < 0 ||
            positions[2 * j + 1] + N > obj_w)
            return NULL;
    oracle_dm *o = calloc(1, sizeof(*o));
    o->N = N; o->n_views = n_views; o->K = K; o->L = L; o->H = obj_h; o->W = obj_w;
    o->pos = malloc(sizeof(int32_t) * 2 * n_views);
    memcpy(o->pos, positions, sizeof(int32_t) * 2 * n_views);
    o->beta = 1; o->a_obj = (real)1e-3; o->a_probe = (real)1e-3; o->eps_f = (real)1e-30;
    size_t NN = (size_t)N * N;
    o->P = malloc(sizeof(cplx) * K * NN);
    o->O = malloc(sizeof(cplx) * L * (size_t)obj_h * obj_w);
    o->psi = malloc(sizeof(cplx) * (size_t)n_views * K * L * NN);
    o->amp = malloc(sizeof(real) * (size_t)n_views * NN);
    if (!o->P || !o->O || !o->psi || !o->amp) return NULL;
    return o;
}

void oracle_destroy(oracle_dm *o)
{
    if (!o) return;
    free(o->pos); free(o->P); free(o->O); free(o->psi); free(o->amp); free(o->errors); free(o);
}

/* which: 0 beta, 1 a_obj, 2 a_probe, 3 eps_f (same order as dm_param in include/dm.h) */
int oracle_set_param(oracle_dm *o, int which, double v)
{
    switch (which) {
    case 0: if (v < 0 || v > 1) return -1; o->beta = (real)v; return 0;
    case 1: if (v < 0) return -1; o->a_obj = (real)v; return 0;
    case 2: if (v < 0) return -1; o->a_probe = (real)v; return 0;
    case 3: if (v < 0) return -1; o->eps_f = (real)v; return 0;
    }
    return -1;
}

/* Inputs are the float32 / complex64 arrays both sides receive, widened here (A20).
 * amp = sqrt(I); psi = P0 * O0|window; alpha frozen from P0, O0 (A8):
 *   alpha_obj   = a_obj   * max_r sum_{j covers r} sum_k |P0_k(r - r_j)|^2
 *   alpha_probe = a_probe * max_r sum_j sum_l |O0_l(r + r_j)|^2                          */
int oracle_set_data(oracle_dm *o, const float *intensities, const float *probe0,
                    const float *object0)
{
    size_t NN = (size_t)o->N * o->N, HW = (size_t)o->H * o->W;
    int N = o->N, K = o->K, L = o->L, W = o->W;
    for (size_t i = 0; i < (size_t)o->n_views * NN; ++i) o->amp[i] = sqrt((real)intensities[i]);
    for (size_t i = 0; i < K * NN; ++i) o->P[i] = (real)probe0[2 * i] + (real)probe0[2 * i + 1] * I;
    for (size_t i = 0; i < L * HW; ++i) o->O[i] = (real)object0[2 * i] + (real)object0[2 * i + 1] * I;
#pragma omp parallel for schedule(static)
    for (int j = 0; j < o->n_views; ++j)
        for (int k = 0; k < K; ++k)
            for (int l = 0; l < L; ++l)
                for (int ry = 0; ry < N; ++ry)
                    for (int rx = 0; rx < N; ++rx)
                        o->psi[(((size_t)j * K + k) * L + l) * NN + (size_t)ry * N + rx] =
                            o->P[k * NN + (size_t)ry * N + rx] *
                            o->O[l * HW + (size_t)(o->pos[2 * j] + ry) * W + o->pos[2 * j + 1] + rx];
    /* frozen regularisers */
    real *den = calloc(HW, sizeof(real));
    for (int j = 0; j < o->n_views; ++j)
        for (int ry = 0; ry < N; ++ry)
            for (int rx = 0; rx < N; ++rx) {
                real s = 0;
                for (int k = 0; k < K; ++k) s += cabs2(o->P[k * NN + (size_t)ry * N + rx]);
                den[(size_t)(o->pos[2 * j] + ry) * W + o->pos[2 * j + 1] + rx] += s;
            }
    real mx = 0;
    for (size_t i = 0; i < HW; ++i) if (den[i] > mx) mx = den[i];
    o->alpha_obj = o->a_obj * mx;
    free(den);
    mx = 0;
    for (int ry = 0; ry < N; ++ry)
        for (int rx = 0; rx < N; ++rx) {
            real s = 0;
            for (int j = 0; j < o->n_views; ++j)
                for (int l = 0; l < L; ++l)
                    s += cabs2(o->O[l * HW + (size_t)(o->pos[2 * j] + ry) * W + o->pos[2 * j + 1] + rx]);
            if (s > mx) mx = s;
        }
    o->alpha_probe = o->a_probe * mx;
    o->has_data = 1;
    o->n_rows = 0;
    return 0;
}

void oracle_get_alphas(const oracle_dm *o, double *out2)
{
    out2[0] = (double)o->alpha_obj; out2[1] = (double)o->alpha_probe;
}

int oracle_iterate(oracle_dm *o, int n_iter)
{
    if (!o->has_data || n_iter < 0) return -1;
    int N = o->N, K = o->K, L = o->L, nv = o->n_views, ncol = 2 + K + L;
    size_t NN = (size_t)N * N, HW = (size_t)o->H * o->W;
    cplx *On = malloc(sizeof(cplx) * L * HW), *Pn = malloc(sizeof(cplx) * K * NN);
    real *acc = malloc(sizeof(real) * 4 * nv);
    for (int it = 0; it < n_iter; ++it) {
        /* A: every view independently */
#pragma omp parallel for schedule(dynamic, 1)
        for (int j = 0; j < nv; ++j) {
            real a[4] = {0, 0, 0, 0};
            oracle_view_update(N, K, L, (real *)o->P, (real *)o->O, o->H, o->W, o->pos[2 * j],
                               o->pos[2 * j + 1], (real *)(o->psi + (size_t)j * K * L * NN),
                               o->amp + (size_t)j * NN, o->beta, o->eps_f, a, 0);
            memcpy(acc + 4 * j, a, sizeof(a));
        }
        real eF_num = 0, eF_den = 0, ep_num = 0, ep_den = 0;   /* fixed order: j ascending */
        for (int j = 0; j < nv; ++j) {
            eF_num += acc[4 * j]; eF_den += acc[4 * j + 1];
            ep_num += acc[4 * j + 2]; ep_den += acc[4 * j + 3];
        }
        /* B then C */
        oracle_object_update(N, nv, K, L, o->H, o->W, o->pos, (real *)o->P, (real *)o->psi,
                             (real *)o->O, o->alpha_obj, (real *)On);
        oracle_probe_update(N, nv, K, L, o->H, o->W, o->pos, (real *)On, (real *)o->psi,
                            (real *)o->P, o->alpha_probe, (real *)Pn);
        /* D */
        if (o->n_rows == o->cap_rows) {
            o->cap_rows = o->cap_rows ? 2 * o->cap_rows : 64;
            o->errors = realloc(o->errors, sizeof(double) * ncol * o->cap_rows);
        }
        double *row = o->errors + (size_t)ncol * o->n_rows++;
        row[0] = eF_den > 0 ? sqrt((double)(eF_num / eF_den)) : 0;
        row[1] = ep_den > 0 ? sqrt((double)(ep_num / ep_den)) : 0;
        for (int k = 0; k < K; ++k)
            row[2 + k] = (double)oracle_rel_change(NN, (real *)(Pn + k * NN), (real *)(o->P + k * NN));
        for (int l = 0; l < L; ++l)
            row[2 + K + l] = (double)oracle_rel_change(HW, (real *)(On + l * HW), (real *)(o->O + l * HW));
        memcpy(o->P, Pn, sizeof(cplx) * K * NN);
        memcpy(o->O, On, sizeof(cplx) * L * HW);
    }
    free(On); free(Pn); free(acc);
    return 0;
}

void oracle_get_probe(const oracle_dm *o, real *out)
{ memcpy(out, o->P, sizeof(cplx) * o->K * (size_t)o->N * o->N); }
void oracle_get_object(const oracle_dm *o, real *out)
{ memcpy(out, o->O, sizeof(cplx) * o->L * (size_t)o->H * o->W); }
void oracle_get_psi(const oracle_dm *o, real *out)
{ memcpy(out, o->psi, sizeof(cplx) * (size_t)o->n_views * o->K * o->L * o->N * o->N); }
/* NULL = keep.  Does not touch amp, the frozen alphas or the error table. */
void oracle_set_state(oracle_dm *o, const real *P, const real *O, const real *psi)
{
    if (P) memcpy(o->P, P, sizeof(cplx) * o->K * (size_t)o->N * o->N);
    if (O) memcpy(o->O, O, sizeof(cplx) * o->L * (size_t)o->H * o->W);
    if (psi) memcpy(o->psi, psi, sizeof(cplx) * (size_t)o->n_views * o->K * o->L * o->N * o->N);
}
int oracle_get_errors(const oracle_dm *o, double *out, int max_rows)
{
    int n = o->n_rows < max_rows ? o->n_rows : max_rows;
    memcpy(out, o->errors, sizeof(double) * (2 + o->K + o->L) * (size_t)n);
    return n;
}
int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
void oracle_set_num_threads(int n)
{
#ifdef _OPENMP
    omp_set_num_threads(n);
#else
    (void)n;
#endif
}
int oracle_real_bytes(void) { return (int)sizeof(real); }

/* ------------------------------------------------ view-range entry points ----
 * The same steps as oracle_iterate, cut along the view axis so that a caller can stream a
 * problem whose psi (complex128: 32 GiB for BASELINE.json config 3) does not fit host memory.
 * Nothing new is computed: eq. (6) / eq. (5) are sums over the views j, and a sum
 * carried in a caller-held accumulator over consecutive ranges [j0, j1) performs exactly the additions
 * of oracle_object_update / oracle_probe_update in exactly their order (j ascending, then k resp. l
 * ascending: readings A3, A15 of DESIGN.md), so the results are bit-identical to the monolithic
 * functions for any split -- which tests/test_oracle_dm.py requires.  The denominators do not depend on
 * the mode of the numerator (A15), so one [H][W] resp. [N][N] array serves all modes.              */

/* Step A on views j0 <= j < j1 (each one oracle_view_update, as in oracle_iterate).
 * psi_range_io [j1-j0][K][L][N][N] in/out, amp_range [j1-j0][N][N], acc_out [j1-j0][4].        */
void oracle_views_update(int N, int j0, int j1, int K, int L, const real *P_in, const real *O_in,
                         int obj_h, int obj_w, const int32_t *positions, real *psi_range_io,
                         const real *amp_range, real beta, real eps, real *acc_out)
{
    size_t NN = (size_t)N * N;
#pragma omp parallel for schedule(dynamic, 1)
    for (int j = j0; j < j1; ++j) {
        real a[4] = {0, 0, 0, 0};
        oracle_view_update(N, K, L, P_in, O_in, obj_h, obj_w, positions[2 * j], positions[2 * j + 1],
                           psi_range_io + 2 * (size_t)(j - j0) * K * L * NN,
                           amp_range + (size_t)(j - j0) * NN, beta, eps, a, 0);
        memcpy(acc_out + 4 * (size_t)(j - j0), a, sizeof(a));
    }
}

/* eq. (6) numerator / denominator of views j0 <= j < j1 added onto num (cplx [L][H][W]) and den
 * (real [H][W]); the caller zeroes both before the first range.  positions = the FULL list.     */
void oracle_object_accumulate(int N, int j0, int j1, int K, int L, int obj_h, int obj_w,
                              const int32_t *positions, const real *P_in, const real *psi_range_in,
                              real *num_io, real *den_io)
{
    const cplx *P = (const cplx *)P_in, *psi = (const cplx *)psi_range_in;
    cplx *numa = (cplx *)num_io;
    size_t NN = (size_t)N * N, HW = (size_t)obj_h * obj_w;
#pragma omp parallel for schedule(static)
    for (int y = 0; y < obj_h; ++y)
        for (int x = 0; x < obj_w; ++x)
            for (int l = 0; l < L; ++l) {
                size_t o = (size_t)y * obj_w + x;
                cplx num = numa[l * HW + o]; real den = den_io[o];
                for (int j = j0; j < j1; ++j) {
                    int ry = y - positions[2 * j], rx = x - positions[2 * j + 1];
                    if (ry < 0 || ry >= N || rx < 0 || rx >= N) continue;
                    size_t r = (size_t)ry * N + rx;
                    for (int k = 0; k < K; ++k) {
                        cplx p = P[k * NN + r];
                        num += conj(p) * psi[(((size_t)(j - j0) * K + k) * L + l) * NN + r];
                        den += cabs2(p);
                    }
                }
                numa[l * HW + o] = num;
                if (l == L - 1) den_io[o] = den;    /* every l walks the same den sequence: store it once */
            }
}

/* the quotient of eq. (6) with the inertial term (A8), as in oracle_object_update */
void oracle_object_finish(int L, int obj_h, int obj_w, const real *num_in, const real *den_in,
                          const real *O_old_in, real alpha, real *O_new_out)
{
    const cplx *num = (const cplx *)num_in, *Oo = (const cplx *)O_old_in;
    cplx *On = (cplx *)O_new_out;
    size_t HW = (size_t)obj_h * obj_w;
    for (int l = 0; l < L; ++l)
        for (size_t o = 0; o < HW; ++o) {
            real den = den_in[o];
            On[l * HW + o] = (alpha + den > 0) ? (alpha * Oo[l * HW + o] + num[l * HW + o]) / (alpha + den)
                                               : Oo[l * HW + o];
        }
}

/* eq. (5) numerator / denominator of views j0 <= j < j1 added onto num (cplx [K][N][N]) and den
 * (real [N][N]); O is the NEW object (A3).                                                      */
void oracle_probe_accumulate(int N, int j0, int j1, int K, int L, int obj_h, int obj_w,
                             const int32_t *positions, const real *O_in, const real *psi_range_in,
                             real *num_io, real *den_io)
{
    const cplx *O = (const cplx *)O_in, *psi = (const cplx *)psi_range_in;
    cplx *numa = (cplx *)num_io;
    size_t NN = (size_t)N * N, HW = (size_t)obj_h * obj_w;
#pragma omp parallel for schedule(static)
    for (int ry = 0; ry < N; ++ry)
        for (int rx = 0; rx < N; ++rx)
            for (int k = 0; k < K; ++k) {
                size_t r = (size_t)ry * N + rx;
                cplx num = numa[k * NN + r]; real den = den_io[r];
                for (int j = j0; j < j1; ++j)
                    for (int l = 0; l < L; ++l) {
                        cplx o = O[l * HW + (size_t)(positions[2 * j] + ry) * obj_w +
                                   positions[2 * j + 1] + rx];
                        num += conj(o) * psi[(((size_t)(j - j0) * K + k) * L + l) * NN + r];
                        den += cabs2(o);
                    }
                numa[k * NN + r] = num;
                if (k == K - 1) den_io[r] = den;
            }
}

void oracle_probe_finish(int N, int K, const real *num_in, const real *den_in, const real *P_old_in,
                         real alpha, real *P_new_out)
{
    const cplx *num = (const cplx *)num_in, *Po = (const cplx *)P_old_in;
    cplx *Pn = (cplx *)P_new_out;
    size_t NN = (size_t)N * N;
    for (int k = 0; k < K; ++k)
        for (size_t r = 0; r < NN; ++r) {
            real den = den_in[r];
            Pn[k * NN + r] = (alpha + den > 0) ? (alpha * Po[k * NN + r] + num[k * NN + r]) / (alpha + den)
                                               : Po[k * NN + r];
        }
}

/* The frozen regularisers of oracle_set_data (A8) without a state object: the same two loops.
 * P0 cplx [K][N][N], O0 cplx [L][H][W]; out2 = (alpha_obj, alpha_probe).                        */
void oracle_frozen_alphas(int N, int n_views, int K, int L, int obj_h, int obj_w,
                          const int32_t *positions, const real *P0_in, const real *O0_in,
                          real a_obj, real a_probe, double *out2)
{
    const cplx *P = (const cplx *)P0_in, *O = (const cplx *)O0_in;
    size_t NN = (size_t)N * N, HW = (size_t)obj_h * obj_w;
    real *den = calloc(HW, sizeof(real));
    for (int j = 0; j < n_views; ++j)
        for (int ry = 0; ry < N; ++ry)
            for (int rx = 0; rx < N; ++rx) {
                real s = 0;
                for (int k = 0; k < K; ++k) s += cabs2(P[k * NN + (size_t)ry * N + rx]);
                den[(size_t)(positions[2 * j] + ry) * obj_w + positions[2 * j + 1] + rx] += s;
            }
    real mx = 0;
    for (size_t i = 0; i < HW; ++i) if (den[i] > mx) mx = den[i];
    out2[0] = (double)(a_obj * mx);
    free(den);
    mx = 0;
    for (int ry = 0; ry < N; ++ry)
        for (int rx = 0; rx < N; ++rx) {
            real s = 0;
            for (int j = 0; j < n_views; ++j)
                for (int l = 0; l < L; ++l)
                    s += cabs2(O[l * HW + (size_t)(positions[2 * j] + ry) * obj_w + positions[2 * j + 1] + rx]);
            if (s > mx) mx = s;
        }
    out2[1] = (double)(a_probe * mx);
}
