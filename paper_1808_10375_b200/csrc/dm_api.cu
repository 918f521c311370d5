// dm_api.cu -- the C ABI of include/dm.h: host plan (integer tables, workspace carving),
// launch orchestration of one DM iteration, getters.  No torch types, no exceptions.
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/dm.h"
#include "dm_kernels.cuh"
#include "dm_fp64.cuh"

namespace {

constexpr size_t ALIGN = 256;
constexpr int ERR_ROWS_CAP = 16384;
constexpr size_t SCRATCH_TARGET = 48u << 20;     // staged path: spectra of one chunk stay in L2
constexpr int COLS_SW = 8;                        // staged path: spectrum columns per CTA
constexpr int PROF_MAX_ITERS = 4096;

thread_local std::string g_create_error;

size_t align_up(size_t x) { return (x + ALIGN - 1) / ALIGN * ALIGN; }

} // namespace

struct dm_plan {
    int N, n_views, K, L, M, H, W;
    std::vector<int32_t> pos;            // (y0,x0)
    std::vector<int32_t> tile_ptr, tile_views;
    int nty, ntx;
    std::vector<int32_t> rev;            // digit reversal of the FFT passes (paths 1, 2)
    std::vector<int32_t> spec;           // spectrum layout of the chosen path: storage position -> ky*N + kx
    std::vector<float> tw;               // N complex twiddles
    double beta, a_obj, a_probe, eps_f;
    int path_req, path;                  // requested / chosen (1 staged, 2 fused, 3 register-resident)
    int reg_grid;                        // path 3: number of persistent CTAs (multiple of M)
    bool reg_sw;                         // path 3: software group barrier instead of a hardware cluster
    int *reg_gbar;                       // path 3: [reg_cap] group barrier counters (+ 1 spare word)
    int reg_cap;                         // path 3: upper bound on resident CTAs (2 per SM)
    // path 4 (dm_warpfft.cuh): ring slots, phase lag (views), tasks per view and phase, persistent CTAs
    int wf_S, wf_D, wf_nA, wf_nB, wf_nC, wf_grid, wf_nw;
    int wf_lag_req;                      // 0 = derive the lag from the task counts
    int *wf_cnt;                         // [1 + 3 n_views] queue counter, cntA, cntB, cntC
    float2 *wf_tw_d;                     // [N/32][32] stage-1 twiddles
    // probe reduction geometry
    int prb_blocks, prb_chunks, prb_chunk_len, fin_blocks;
    // staged geometry
    int chunk_views;
    // workspace
    void *ws;
    size_t ws_bytes, need_bytes;
    float2 *psi, *Pbuf[2], *Obuf[2], *pnum, *scratch, *tw_d;
    float *amp, *pden, *den_tmp, *alphas, *partA, *partB, *partP, *partO;
    int2 *pos_d;
    int *tile_ptr_d, *tile_views_d, *spec_d;
    float2 *wy_d, *wx_d;                 // path 3 twiddle tables
    float4 *sbuf;                        // path 3 mode-sum exchange (L2 resident)
    double *errors;
    double *mode_pow;                    // [K + L] scratch of dm_get_mode_power
    float *stage_I;
    float2 *stage_P, *stage_O;
    int curP, curO;
    int nA, nB;                          // counts of (num,den) pairs in partA / partB (staged)
    bool has_data;
    int rows;
    // optional per-phase timing (dm_plan_set_profiling)
    bool profiling;
    std::vector<cudaEvent_t> ev;         // 5 events per profiled iteration
    int ev_iters;
    // dm_solve_host: the intensities travel on a second stream, in chunks, under the set-up kernels
    cudaStream_t copy_st;
    cudaEvent_t ev_begin, ev_chunk[8];
    bool copy_ready;
    // DM_PARAM_PRECISION = 1: the FP64 validation mode (dm_fp64.cuh)
    int precision;
    double2 *psi64, *scr64, *P64[2], *O64[2], *tw64;
    double *amp64, *den64, *alphas64, *partF64, *partS64, *partP64, *partO64;
    int tables_path;                     // path whose tables / twiddles are on the device (0: none)
    int sms;                             // SM count of the device (148 until a CUDA call could ask)
    int max_list;                        // longest coverage list (object_gather_kernel batches it by OBJ_NT)
    mutable std::string err;
};

namespace {

dm_status fail(const dm_plan *p, dm_status s, const char *fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    if (p) p->err = buf; else g_create_error = buf;
    return s;
}

#define CU(call)                                                                              \
    do {                                                                                      \
        cudaError_t e_ = (call);                                                              \
        if (e_ != cudaSuccess) return fail(plan, DM_ERR_CUDA, "%s: %s", #call, cudaGetErrorString(e_)); \
    } while (0)

template <int N> void fill_rev(std::vector<int32_t> &rev)
{
    rev.resize(N);
    for (int p = 0; p < N; ++p) rev[p] = dmfft::digit_reverse<N>(p);
}

void build_tables(dm_plan *p)
{
    const int N = p->N, TH = OBJ_TH, TW = OBJ_TW;
    p->nty = (p->H + TH - 1) / TH;
    p->ntx = (p->W + TW - 1) / TW;
    const int nt = p->nty * p->ntx;
    std::vector<int32_t> cnt(nt + 1, 0);
    for (int j = 0; j < p->n_views; ++j) {
        const int y0 = p->pos[2 * j], x0 = p->pos[2 * j + 1];
        for (int ty = y0 / TH; ty <= (y0 + N - 1) / TH; ++ty)
            for (int tx = x0 / TW; tx <= (x0 + N - 1) / TW; ++tx) cnt[ty * p->ntx + tx + 1]++;
    }
    for (int t = 0; t < nt; ++t) cnt[t + 1] += cnt[t];
    p->tile_ptr = cnt;
    p->max_list = 0;
    for (int t = 0; t < nt; ++t) p->max_list = std::max(p->max_list, cnt[t + 1] - cnt[t]);
    p->tile_views.assign((size_t)cnt[nt], 0);
    std::vector<int32_t> fill(cnt.begin(), cnt.end() - 1);
    for (int j = 0; j < p->n_views; ++j) {     // j ascending -> every list ascending
        const int y0 = p->pos[2 * j], x0 = p->pos[2 * j + 1];
        for (int ty = y0 / TH; ty <= (y0 + N - 1) / TH; ++ty)
            for (int tx = x0 / TW; tx <= (x0 + N - 1) / TW; ++tx) p->tile_views[fill[ty * p->ntx + tx]++] = j;
    }
    switch (N) {
    case 64: fill_rev<64>(p->rev); break;
    case 128: fill_rev<128>(p->rev); break;
    case 256: fill_rev<256>(p->rev); break;
    default: fill_rev<512>(p->rev); break;
    }
    p->tw.resize(2 * (size_t)N);
    for (int n = 0; n < N; ++n) {
        const double ang = -2.0 * M_PI * (double)n / (double)N;
        p->tw[2 * n] = (float)std::cos(ang);
        p->tw[2 * n + 1] = (float)std::sin(ang);
    }
}

void plan_geometry(dm_plan *p)
{
    const size_t NN = (size_t)p->N * p->N;
    p->prb_blocks = (int)((NN / 2 + PRB_NT - 1) / PRB_NT);
    int chunks = (p->sms * 16 + p->prb_blocks - 1) / p->prb_blocks;     // ~16 CTAs per SM in flight
    if (chunks > p->n_views) chunks = p->n_views;
    if (chunks < 1) chunks = 1;
    p->prb_chunk_len = (p->n_views + chunks - 1) / chunks;
    p->prb_chunks = (p->n_views + p->prb_chunk_len - 1) / p->prb_chunk_len;
    p->fin_blocks = (int)((NN + 255) / 256);
    p->reg_cap = 2 * p->sms;
    const size_t per_view = (size_t)p->M * NN * sizeof(float2);
    size_t cv = SCRATCH_TARGET / per_view;
    if (cv < 1) cv = 1;
    if (cv > (size_t)p->n_views) cv = p->n_views;
    p->chunk_views = (int)cv;
    // path 4: a CTA task = 8 row groups (phases A, C) or 8 / M column groups x M modes (phase B)
    const int G = 1024 / p->N, NG = p->N / G;
    p->wf_nw = p->M == 1 ? 2 : p->M;                 // warps per CTA
    const int GPT = p->wf_nw / p->M;
    p->wf_nA = (p->M * NG + p->wf_nw - 1) / p->wf_nw;
    p->wf_nC = p->wf_nA;
    p->wf_nB = (NG + GPT - 1) / GPT;
    const int T = p->wf_nA + p->wf_nB + p->wf_nC;
    // lag: a phase starts on a view once ~1.6 x (resident CTAs) tasks have been queued behind its inputs
    // (measured on B200 at the end of round 1: c3 is fastest at 3-4 views, c4 at 2; a longer lag only pushes psi out of L2)
    const int resident = p->sms * (16 / p->wf_nw);
    int D = p->wf_lag_req > 0 ? p->wf_lag_req : (int)((1.6 * resident + T - 1) / T);
    if (D < 1) D = 1;
    p->wf_D = D;
    p->wf_S = 2 * D + 4;
    if (p->wf_S > p->n_views) p->wf_S = p->n_views;
    if (p->wf_S <= 2 * D) p->wf_S = 2 * D + 1;       // keeps "A(v) waits for C(v - S)" behind it in the queue
}

// carve (or, with base == nullptr, just measure) the workspace
size_t carve(dm_plan *p, unsigned char *base)
{
    size_t off = 0;
    auto take = [&](size_t bytes) -> void * {
        void *r = base ? base + off : nullptr;
        off += align_up(bytes);
        return r;
    };
    const size_t NN = (size_t)p->N * p->N, HW = (size_t)p->H * p->W;
    const size_t MV = (size_t)p->n_views * p->M;
    const int rows_tiles = p->N / (4096 / p->N);                         // row tiles per frame (staged)
    p->nA = p->n_views * (p->N / COLS_SW);
    p->nB = (int)(MV * rows_tiles);

    p->psi = (float2 *)take(MV * NN * sizeof(float2));
    p->amp = (float *)take((size_t)p->n_views * NN * sizeof(float));
    for (int i = 0; i < 2; ++i) p->Pbuf[i] = (float2 *)take(p->K * NN * sizeof(float2));
    for (int i = 0; i < 2; ++i) p->Obuf[i] = (float2 *)take(p->L * HW * sizeof(float2));
    p->pnum = (float2 *)take((size_t)p->prb_chunks * p->K * NN * sizeof(float2));
    p->pden = (float *)take((size_t)p->prb_chunks * NN * sizeof(float));
    p->den_tmp = (float *)take((HW > NN ? HW : NN) * sizeof(float));
    p->alphas = (float *)take(2 * sizeof(float));
    size_t nA = (size_t)p->nA * 2 > MV * 4 ? (size_t)p->nA * 2 : MV * 4;
    if (nA < (size_t)p->reg_cap * 4) nA = (size_t)p->reg_cap * 4;
    if (nA < (size_t)p->n_views * p->wf_nB * 2) nA = (size_t)p->n_views * p->wf_nB * 2;
    size_t nB = (size_t)p->nB * 2;
    if (nB < (size_t)p->n_views * p->wf_nC * 2) nB = (size_t)p->n_views * p->wf_nC * 2;
    p->partA = (float *)take(nA * sizeof(float));
    p->partB = (float *)take(nB * sizeof(float));
    p->partP = (float *)take((size_t)p->fin_blocks * p->K * 2 * sizeof(float));
    p->partO = (float *)take((size_t)p->nty * p->ntx * p->L * 2 * sizeof(float));
    p->pos_d = (int2 *)take((size_t)p->n_views * sizeof(int2));
    p->tile_ptr_d = (int *)take(p->tile_ptr.size() * sizeof(int));
    p->tile_views_d = (int *)take((p->tile_views.size() + 1) * sizeof(int));
    p->spec_d = (int *)take(NN * sizeof(int));
    p->wy_d = (float2 *)take(128 * sizeof(float2));
    p->wx_d = (float2 *)take(128 * sizeof(float2));
    p->sbuf = (float4 *)take(p->N == 128 ? (size_t)2 * p->reg_cap * 8 * dmreg::RNT * sizeof(float4) : 0);
    p->reg_gbar = (int *)take(((size_t)p->reg_cap + 1) * sizeof(int));
    p->tw_d = (float2 *)take(p->N * sizeof(float2));
    p->mode_pow = (double *)take((size_t)(p->K + p->L) * sizeof(double));
    p->errors = (double *)take((size_t)ERR_ROWS_CAP * (2 + p->K + p->L) * sizeof(double));
    {
        size_t sc = (size_t)p->chunk_views * p->M * NN, ring = (size_t)p->wf_S * p->M * NN;
        p->scratch = (float2 *)take((sc > ring ? sc : ring) * sizeof(float2));
    }
    p->wf_cnt = (int *)take((1 + 3 * (size_t)p->n_views) * sizeof(int));
    p->wf_tw_d = (float2 *)take((size_t)p->N * sizeof(float2));
    if (p->precision == 1) {
        p->psi64 = (double2 *)take(MV * NN * sizeof(double2));
        p->scr64 = (double2 *)take(MV * NN * sizeof(double2));
        for (int i = 0; i < 2; ++i) p->P64[i] = (double2 *)take(p->K * NN * sizeof(double2));
        for (int i = 0; i < 2; ++i) p->O64[i] = (double2 *)take(p->L * HW * sizeof(double2));
        p->tw64 = (double2 *)take((size_t)p->N / 2 * sizeof(double2));
        p->amp64 = (double *)take((size_t)p->n_views * NN * sizeof(double));
        p->den64 = (double *)take((HW > NN ? HW : NN) * sizeof(double));
        p->alphas64 = (double *)take(2 * sizeof(double));
        p->partF64 = (double *)take((size_t)p->n_views * (NN / 256) * 2 * sizeof(double));
        p->partS64 = (double *)take(MV * p->N * 2 * sizeof(double));
        p->partP64 = (double *)take((size_t)(NN / 256) * p->K * 2 * sizeof(double));
        p->partO64 = (double *)take((size_t)p->nty * p->ntx * p->L * 2 * sizeof(double));
    }
    p->stage_I = (float *)take((size_t)p->n_views * NN * sizeof(float));
    p->stage_P = (float2 *)take(p->K * NN * sizeof(float2));
    p->stage_O = (float2 *)take(p->L * HW * sizeof(float2));
    return off;
}

PsiArgs psi_args(const dm_plan *p)
{
    PsiArgs a;
    memset(&a, 0, sizeof a);
    a.n_views = p->n_views; a.K = p->K; a.L = p->L; a.H = p->H; a.W = p->W;
    a.pos = p->pos_d; a.P = p->Pbuf[p->curP]; a.O = p->Obuf[p->curO];
    a.psi = p->psi; a.amp = p->amp; a.tw = p->tw_d;
    a.beta = (float)p->beta; a.eps = (float)p->eps_f;
    a.part = p->partA; a.part2 = p->partB; a.scratch = p->scratch;
    return a;
}

// Every launch_* below takes `prepare`: true = called once per plan from dm_set_data on the plan's device to
// opt the kernel in to its dynamic shared memory (a per-device function attribute) and to size the persistent
// grids from occupancy queries; nothing is launched then.
template <int N, int NT> dm_status launch_fused(dm_plan *plan, cudaStream_t st, bool prepare)
{
    const size_t smem = (size_t)N * N * (sizeof(float2) + sizeof(float)) + N * sizeof(float2);
    if (prepare) {
        CU(cudaFuncSetAttribute(fused_frame_kernel<N, NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        return DM_OK;
    }
    PsiArgs a = psi_args(plan);
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof cfg);
    cfg.gridDim = dim3((unsigned)(plan->n_views * plan->M));
    cfg.blockDim = dim3(NT);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)plan->M;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    CU(cudaLaunchKernelEx(&cfg, fused_frame_kernel<N, NT>, a));
    return DM_OK;
}

template <int N> dm_status launch_staged(dm_plan *plan, cudaStream_t st, bool prepare)
{
    constexpr int ROWS = 4096 / N, NT = 256, SW = COLS_SW;
    const size_t smem = (size_t)plan->M * N * SW * sizeof(float2);
    if (prepare) {
        if (smem > 200 * 1024)
            return fail(plan, DM_ERR_UNSUPPORTED, "staged path: %d modes of N = %d need %zu bytes of shared memory per CTA", plan->M, N, smem);
        CU(cudaFuncSetAttribute(cols_mod_kernel<N, SW, NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
        return DM_OK;
    }
    PsiArgs a = psi_args(plan);
    for (int v0 = 0; v0 < plan->n_views; v0 += plan->chunk_views) {
        const int nv = plan->n_views - v0 < plan->chunk_views ? plan->n_views - v0 : plan->chunk_views;
        a.view0 = v0;
        a.n_chunk = nv;
        const unsigned row_tiles = (unsigned)(nv * plan->M * (N / ROWS));
        rows_fwd_kernel<N, ROWS, NT><<<row_tiles, NT, 0, st>>>(a);
        cols_mod_kernel<N, SW, NT><<<dim3(N / SW, nv), NT, smem, st>>>(a);
        rows_inv_kernel<N, ROWS, NT><<<row_tiles, NT, 0, st>>>(a);
    }
    CU(cudaGetLastError());
    return DM_OK;
}

// path 3: persistent register-resident kernel, cluster = the M mode frames of a view
template <int MT> dm_status launch_regfft_t(dm_plan *plan, cudaStream_t st, bool query_only)
{
    auto kern = dmreg::regfft128_kernel<MT>;
    if (query_only) CU(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, dmreg::REG_SMEM_V1));
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof cfg);
    cfg.blockDim = dim3(dmreg::RNT);
    cfg.dynamicSmemBytes = dmreg::REG_SMEM_V1;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)plan->M;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = plan->M > 1 ? 1 : 0;
    if (query_only) {
        int ncl = 0, dev = 0, sms = 0, per = 0;
        CU(cudaGetDevice(&dev));
        CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per, kern, dmreg::RNT, dmreg::REG_SMEM_V1));
        plan->reg_sw = false;
        if (plan->M > 1) {
            cfg.gridDim = dim3((unsigned)plan->M);
            CU(cudaOccupancyMaxActiveClusters(&ncl, kern, &cfg));
            // a cluster of M can strand SMs (M = 4: 132 of 148 on B200); then the M CTAs of a view
            // synchronise through a counter in L2 instead and the grid fills every SM
            const int ncl_sw = sms * per / plan->M;
            if (ncl_sw > ncl) { ncl = ncl_sw; plan->reg_sw = true; }
        } else {
            ncl = sms * per;
        }
        if (ncl < 1) return fail(plan, DM_ERR_CUDA, "register-resident kernel: no cluster of %d CTAs fits", plan->M);
        if (ncl > plan->n_views) ncl = plan->n_views;
        if (ncl * plan->M > plan->reg_cap) ncl = plan->reg_cap / plan->M;
        plan->reg_grid = ncl * plan->M;
        return DM_OK;
    }
    dmreg::RegArgs a;
    memset(&a, 0, sizeof a);
    a.n_views = plan->n_views; a.K = plan->K; a.L = plan->L; a.H = plan->H; a.W = plan->W;
    a.pos = plan->pos_d; a.P = plan->Pbuf[plan->curP]; a.O = plan->Obuf[plan->curO];
    a.psi = plan->psi; a.amp = plan->amp; a.wy = plan->wy_d; a.wx = plan->wx_d;
    a.sbuf = plan->sbuf; a.part = plan->partA;
    a.beta = (float)plan->beta; a.eps = (float)plan->eps_f;
    cfg.gridDim = dim3((unsigned)plan->reg_grid);
    if (plan->reg_sw) {
        a.gbar = plan->reg_gbar;
        CU(cudaMemsetAsync(plan->reg_gbar, 0, (size_t)plan->reg_cap * sizeof(int), st));
        at[0].id = cudaLaunchAttributeCooperative;      // all CTAs resident: they wait on one another
        at[0].val.cooperative = 1;
        cfg.numAttrs = 1;
    }
    CU(cudaLaunchKernelEx(&cfg, kern, a));
    return DM_OK;
}

dm_status launch_regfft(dm_plan *plan, cudaStream_t st, bool query_only)
{
    switch (plan->M) {
    case 1: return launch_regfft_t<1>(plan, st, query_only);
    case 2: return launch_regfft_t<2>(plan, st, query_only);
    case 3: return launch_regfft_t<3>(plan, st, query_only);
    case 4: return launch_regfft_t<4>(plan, st, query_only);
    default: return launch_regfft_t<0>(plan, st, query_only);
    }
}

// path 4: persistent task-queue kernel (rows -> columns + modulus -> rows through an L2-resident ring)
template <int N> dm_status launch_wf_t(dm_plan *plan, cudaStream_t st, bool query_only)
{
    auto kern = dmwf::wf_dataflow_kernel<N>;
    const int nt = 32 * plan->wf_nw;
    const int smem = plan->wf_nw * dmwf::WF_XBUF + (N / 32) * 32 * (int)sizeof(float2) + (plan->wf_nw / plan->M) * 4096;
    if (query_only)
        CU(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                dmwf::WF_MAXW * dmwf::WF_XBUF + (N / 32) * 32 * (int)sizeof(float2) + dmwf::WF_MAXW * 4096));
    if (query_only) {
        int dev = 0, sms = 0, per = 0;
        CU(cudaGetDevice(&dev));
        CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per, kern, nt, smem));
        if (per < 1) return fail(plan, DM_ERR_CUDA, "warp-FFT kernel does not fit an SM");
        plan->wf_grid = sms * per;
        return DM_OK;
    }
    dmwf::WfArgs a;
    memset(&a, 0, sizeof a);
    a.n_views = plan->n_views; a.K = plan->K; a.L = plan->L; a.H = plan->H; a.W = plan->W;
    a.pos = plan->pos_d; a.P = plan->Pbuf[plan->curP]; a.O = plan->Obuf[plan->curO];
    a.psi = plan->psi; a.amp = plan->amp; a.tw = plan->wf_tw_d; a.scratch = plan->scratch;
    a.S = plan->wf_S; a.D = plan->wf_D; a.nA = plan->wf_nA; a.nB = plan->wf_nB; a.nC = plan->wf_nC;
    a.queue = plan->wf_cnt; a.cntA = plan->wf_cnt + 1; a.cntB = a.cntA + plan->n_views; a.cntC = a.cntB + plan->n_views;
    a.partF = plan->partA; a.partS = plan->partB;
    a.beta = (float)plan->beta; a.eps = (float)plan->eps_f;
    CU(cudaMemsetAsync(plan->wf_cnt, 0, (1 + 3 * (size_t)plan->n_views) * sizeof(int), st));
    const long long tasks = (long long)(plan->n_views + 2 * plan->wf_D) * (plan->wf_nA + plan->wf_nB + plan->wf_nC);
    const int grid = tasks < plan->wf_grid ? (int)tasks : plan->wf_grid;
    kern<<<grid, nt, smem, st>>>(a);
    CU(cudaGetLastError());
    return DM_OK;
}

dm_status launch_wf(dm_plan *plan, cudaStream_t st, bool query_only)
{
    switch (plan->N) {
    case 64: return launch_wf_t<64>(plan, st, query_only);
    case 128: return launch_wf_t<128>(plan, st, query_only);
    case 256: return launch_wf_t<256>(plan, st, query_only);
    default: return launch_wf_t<512>(plan, st, query_only);
    }
}

dm_status launch_psi_update(dm_plan *plan, cudaStream_t st, bool prepare = false)
{
    if (plan->path == 4) return launch_wf(plan, st, prepare);
    if (plan->path == 3) return launch_regfft(plan, st, prepare);
    if (plan->path == 2) {
        if (plan->N == 64) return launch_fused<64, 256>(plan, st, prepare);
        return launch_fused<128, 512>(plan, st, prepare);
    }
    switch (plan->N) {
    case 64: return launch_staged<64>(plan, st, prepare);
    case 128: return launch_staged<128>(plan, st, prepare);
    case 256: return launch_staged<256>(plan, st, prepare);
    default: return launch_staged<512>(plan, st, prepare);
    }
}

dm_status launch_object(dm_plan *plan, cudaStream_t st, const float2 *P, const float2 *O_old, float2 *O_new,
                        float *den_out)
{
    const int tiles = plan->nty * plan->ntx;
#define OBJ_LAUNCH(KT, LT)                                                                          \
    object_gather_kernel<KT, LT><<<tiles, OBJ_NT, 0, st>>>(plan->N, plan->K, plan->H, plan->W, plan->pos_d, \
        plan->tile_ptr_d, plan->tile_views_d, P, plan->psi, O_old, O_new, plan->alphas, plan->partO, den_out)
    const int KL = plan->K * 16 + plan->L;
    switch (KL) {
    case 1 * 16 + 1: OBJ_LAUNCH(1, 1); break;
    case 2 * 16 + 1: OBJ_LAUNCH(2, 1); break;
    case 3 * 16 + 1: OBJ_LAUNCH(3, 1); break;
    case 4 * 16 + 1: OBJ_LAUNCH(4, 1); break;
    case 1 * 16 + 2: OBJ_LAUNCH(1, 2); break;
    case 2 * 16 + 2: OBJ_LAUNCH(2, 2); break;
    case 4 * 16 + 2: OBJ_LAUNCH(4, 2); break;
    default:
        switch (plan->L) {
        case 1: OBJ_LAUNCH(0, 1); break;
        case 2: OBJ_LAUNCH(0, 2); break;
        case 3: OBJ_LAUNCH(0, 3); break;
        case 4: OBJ_LAUNCH(0, 4); break;
        case 5: OBJ_LAUNCH(0, 5); break;
        case 6: OBJ_LAUNCH(0, 6); break;
        case 7: OBJ_LAUNCH(0, 7); break;
        default: OBJ_LAUNCH(0, 8); break;
        }
    }
#undef OBJ_LAUNCH
    CU(cudaGetLastError());
    return DM_OK;
}

dm_status launch_probe(dm_plan *plan, cudaStream_t st, const float2 *O, const float2 *P_old, float2 *P_new,
                       float *den_out)
{
    const dim3 grid((unsigned)plan->prb_blocks, (unsigned)plan->prb_chunks);
#define PRB_LAUNCH(KT)                                                                              \
    probe_partial_kernel<KT><<<grid, PRB_NT, 0, st>>>(plan->N, plan->L, plan->n_views, plan->prb_chunk_len, \
        plan->H, plan->W, plan->pos_d, O, plan->psi, plan->pnum, plan->pden)
    switch (plan->K) {
    case 1: PRB_LAUNCH(1); break;
    case 2: PRB_LAUNCH(2); break;
    case 3: PRB_LAUNCH(3); break;
    case 4: PRB_LAUNCH(4); break;
    case 5: PRB_LAUNCH(5); break;
    case 6: PRB_LAUNCH(6); break;
    case 7: PRB_LAUNCH(7); break;
    default: PRB_LAUNCH(8); break;
    }
#undef PRB_LAUNCH
    probe_finalize_kernel<<<dim3((unsigned)plan->fin_blocks, (unsigned)plan->K), 256, 0, st>>>(plan->N, plan->K, plan->prb_chunks, plan->pnum, plan->pden,
                                                            P_old, P_new, plan->alphas, plan->partP, den_out);
    CU(cudaGetLastError());
    return DM_OK;
}

// The grids and the reduction geometry follow the SM count of the current device; without a device
// (CPU-only callers of the host tables) the B200's 148 stays.  Re-measures the workspace.
void adopt_device(dm_plan *p)
{
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) {
        cudaGetLastError();
        return;
    }
    if (sms == p->sms) return;
    p->sms = sms;
    plan_geometry(p);
    p->need_bytes = carve(p, nullptr);
}

dm_status check_ready(const dm_plan *plan, bool need_data)
{
    if (!plan) return DM_ERR_INVALID_ARG;
    if (!plan->ws) return fail(plan, DM_ERR_WORKSPACE, "no workspace set");
    if (need_data && !plan->has_data) return fail(plan, DM_ERR_NO_DATA, "dm_set_data has not been called");
    return DM_OK;
}

} // namespace

extern "C" {

dm_status dm_plan_create(dm_plan **out, int N, int n_views, int K, int L, int obj_h, int obj_w,
                         const int32_t *positions)
{
    if (!out) return fail(nullptr, DM_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    if (!positions) return fail(nullptr, DM_ERR_INVALID_ARG, "positions is NULL");
    if (N <= 0 || n_views <= 0 || K <= 0 || L <= 0 || obj_h <= 0 || obj_w <= 0)
        return fail(nullptr, DM_ERR_INVALID_ARG, "sizes must be positive");
    if (N != 64 && N != 128 && N != 256 && N != 512)
        return fail(nullptr, DM_ERR_UNSUPPORTED, "N = %d: supported frame edges are 64, 128, 256, 512", N);
    if ((long long)K * L > 8) return fail(nullptr, DM_ERR_UNSUPPORTED, "K*L = %d > 8", K * L);
    if (obj_w & 1) return fail(nullptr, DM_ERR_UNSUPPORTED, "obj_w = %d must be even", obj_w);
    if ((long long)obj_h * obj_w > (1ll << 30) || (long long)n_views * K * L > (1ll << 24))
        return fail(nullptr, DM_ERR_UNSUPPORTED, "problem too large for 32-bit indexing of tables");
    for (int j = 0; j < n_views; ++j) {
        const int y0 = positions[2 * j], x0 = positions[2 * j + 1];
        if (y0 < 0 || x0 < 0 || (long long)y0 + N > obj_h || (long long)x0 + N > obj_w)
            return fail(nullptr, DM_ERR_OUT_OF_BOUNDS, "view %d window (%d,%d)+%d leaves the %dx%d object", j, y0, x0, N,
                        obj_h, obj_w);
    }
    dm_plan *p = new (std::nothrow) dm_plan();
    if (!p) return fail(nullptr, DM_ERR_INVALID_ARG, "out of host memory");
    p->N = N; p->n_views = n_views; p->K = K; p->L = L; p->M = K * L; p->H = obj_h; p->W = obj_w;
    p->pos.assign(positions, positions + 2 * (size_t)n_views);
    p->beta = 1.0; p->a_obj = 1e-3; p->a_probe = 1e-3; p->eps_f = 1e-30;
    p->path_req = 0; p->path = 0; p->wf_lag_req = 0;
    p->ws = nullptr; p->ws_bytes = 0;
    p->curP = p->curO = 0; p->has_data = false; p->rows = 0;
    p->profiling = false; p->ev_iters = 0; p->copy_ready = false; p->tables_path = 0; p->precision = 0;
    p->sms = 148;
    build_tables(p);
    plan_geometry(p);
    p->need_bytes = carve(p, nullptr);
    *out = p;
    return DM_OK;
}

dm_status dm_plan_set_param(dm_plan *plan, dm_param which, double v)
{
    if (!plan) return DM_ERR_INVALID_ARG;
    if (plan->has_data) return fail(plan, DM_ERR_INVALID_ARG, "parameters must be set before dm_set_data");
    if (!(v == v)) return fail(plan, DM_ERR_INVALID_ARG, "NaN parameter");
    switch (which) {
    case DM_PARAM_BETA: if (v < 0 || v > 1) break; plan->beta = v; return DM_OK;
    case DM_PARAM_ALPHA_OBJ: if (v < 0) break; plan->a_obj = v; return DM_OK;
    case DM_PARAM_ALPHA_PROBE: if (v < 0) break; plan->a_probe = v; return DM_OK;
    case DM_PARAM_EPS_F: if (v < 0) break; plan->eps_f = v; return DM_OK;
    case DM_PARAM_PATH: if (v != 0 && v != 1 && v != 2 && v != 3 && v != 4) break; plan->path_req = (int)v; return DM_OK;
    case DM_PARAM_PRECISION:
        if (v != 0 && v != 1) break;
        if (plan->ws) return fail(plan, DM_ERR_INVALID_ARG, "the precision sizes the workspace: set it before dm_plan_set_workspace");
        plan->precision = (int)v;
        plan->need_bytes = carve(plan, nullptr);
        return DM_OK;
    case DM_PARAM_LAG:
        if (v < 0 || v > 4096 || v != (double)(int)v) break;
        if (plan->ws) return fail(plan, DM_ERR_INVALID_ARG, "the phase lag sizes the workspace: set it before dm_plan_set_workspace");
        plan->wf_lag_req = (int)v;
        plan_geometry(plan);
        plan->need_bytes = carve(plan, nullptr);
        return DM_OK;
    default: return fail(plan, DM_ERR_INVALID_ARG, "unknown parameter %d", (int)which);
    }
    return fail(plan, DM_ERR_INVALID_ARG, "parameter %d: value %g out of range", (int)which, v);
}

dm_status dm_plan_workspace_bytes(dm_plan *plan, size_t *bytes)
{
    if (!plan || !bytes) return DM_ERR_INVALID_ARG;
    if (!plan->ws) adopt_device(plan);
    *bytes = plan->need_bytes;
    return DM_OK;
}

dm_status dm_plan_set_workspace(dm_plan *plan, void *dev, size_t bytes)
{
    if (!plan) return DM_ERR_INVALID_ARG;
    if (!dev) return fail(plan, DM_ERR_INVALID_ARG, "workspace pointer is NULL");
    if ((uintptr_t)dev % ALIGN) return fail(plan, DM_ERR_WORKSPACE, "workspace must be 256-byte aligned");
    adopt_device(plan);
    if (bytes < plan->need_bytes)
        return fail(plan, DM_ERR_WORKSPACE, "workspace of %zu bytes < %zu needed", bytes, plan->need_bytes);
    plan->ws = dev;
    plan->ws_bytes = bytes;
    carve(plan, (unsigned char *)dev);
    plan->has_data = false;
    plan->tables_path = 0;
    return DM_OK;
}

} // extern "C"

namespace {
constexpr int CONV_GRID = 148 * 8;                 // grid-stride conversion kernels: any grid is correct

dm64::Args args64(const dm_plan *p)
{
    dm64::Args a;
    memset(&a, 0, sizeof a);
    a.N = p->N; a.logN = 0;
    while ((1 << a.logN) < p->N) ++a.logN;
    a.n_views = p->n_views; a.K = p->K; a.L = p->L; a.H = p->H; a.W = p->W;
    a.pos = p->pos_d; a.P = p->P64[p->curP]; a.O = p->O64[p->curO];
    a.psi = p->psi64; a.scratch = p->scr64; a.amp = p->amp64; a.tw = p->tw64;
    a.beta = p->beta; a.eps = p->eps_f;
    a.partF = p->partF64; a.partS = p->partS64;
    return a;
}

dm_status launch_object64(dm_plan *plan, cudaStream_t st, const double2 *P, const double2 *O_old, double2 *O_new, double *den_out)
{
    dm64::object64_kernel<<<plan->nty * plan->ntx, OBJ_TH * OBJ_TW, 0, st>>>(
        plan->N, plan->K, plan->L, plan->H, plan->W, OBJ_TH, OBJ_TW, plan->pos_d, plan->tile_ptr_d, plan->tile_views_d, P,
        plan->psi64, O_old, O_new, plan->alphas64, plan->partO64, den_out);
    CU(cudaGetLastError());
    return DM_OK;
}

dm_status launch_probe64(dm_plan *plan, cudaStream_t st, const double2 *O, const double2 *P_old, double2 *P_new, double *den_out)
{
    const size_t NN = (size_t)plan->N * plan->N;
    dm64::probe64_kernel<<<dim3((unsigned)(NN / 256), (unsigned)plan->K), 256, 0, st>>>(
        plan->N, plan->K, plan->L, plan->n_views, plan->H, plan->W, plan->pos_d, O, plan->psi64, P_old, P_new,
        plan->alphas64, plan->partP64, den_out);
    CU(cudaGetLastError());
    return DM_OK;
}

// FP64 mode: state from float32 / complex64 inputs (widened exactly), psi = P0 * O0, frozen regularisers
dm_status set_data64(dm_plan *plan, const float *intensities, const float *probe0, const float *object0, cudaStream_t st)
{
    const size_t NN = (size_t)plan->N * plan->N, HW = (size_t)plan->H * plan->W;
    std::vector<double> tw((size_t)plan->N);
    for (int n = 0; n < plan->N / 2; ++n) {
        const double ang = -2.0 * M_PI * (double)n / (double)plan->N;
        tw[2 * n] = std::cos(ang);
        tw[2 * n + 1] = std::sin(ang);
    }
    CU(cudaMemcpyAsync(plan->tw64, tw.data(), tw.size() * sizeof(double), cudaMemcpyHostToDevice, st));
    CU(cudaStreamSynchronize(st));
    plan->curP = plan->curO = 0;
    dm64::f2d_kernel<<<CONV_GRID, 256, 0, st>>>(probe0, (double *)plan->P64[0], 2 * plan->K * NN, 0);
    dm64::f2d_kernel<<<CONV_GRID, 256, 0, st>>>(object0, (double *)plan->O64[0], 2 * plan->L * HW, 0);
    dm64::f2d_kernel<<<CONV_GRID, 256, 0, st>>>(intensities, plan->amp64, (size_t)plan->n_views * NN, 1);
    CU(cudaMemsetAsync(plan->alphas64, 0, 2 * sizeof(double), st));
    dm64::psi_init64_kernel<<<dim3((unsigned)((NN + 1023) / 1024), (unsigned)(plan->n_views * plan->M)), 256, 0, st>>>(
        plan->N, plan->K, plan->L, plan->H, plan->W, plan->pos_d, plan->P64[0], plan->O64[0], plan->psi64);
    CU(cudaGetLastError());
    dm_status s = launch_object64(plan, st, plan->P64[0], plan->O64[0], plan->O64[1], plan->den64);
    if (s != DM_OK) return s;
    dm64::max_scale64_kernel<<<1, 1024, 0, st>>>(plan->den64, HW, plan->a_obj, plan->alphas64);
    s = launch_probe64(plan, st, plan->O64[0], plan->P64[0], plan->P64[1], plan->den64);
    if (s != DM_OK) return s;
    dm64::max_scale64_kernel<<<1, 1024, 0, st>>>(plan->den64, NN, plan->a_probe, plan->alphas64 + 1);
    CU(cudaGetLastError());
    return DM_OK;
}

// FP64 mode: one DM iteration (order of DESIGN.md §1: psi update, object, probe, error row)
dm_status iterate64(dm_plan *plan, cudaStream_t st)
{
    const int N = plan->N;
    const size_t NN = (size_t)N * N;
    const unsigned lines = (unsigned)((size_t)plan->n_views * plan->M * N);
    const size_t sm_rows = (size_t)N * sizeof(double2) + (size_t)N * sizeof(double), sm_cols = (size_t)N * sizeof(double2);
    dm64::Args a = args64(plan);
    dm64::rows64_kernel<true><<<lines, N / 2, sm_rows, st>>>(a);
    dm64::cols64_kernel<false><<<lines, N / 2, sm_cols, st>>>(a);
    dm64::modulus64_kernel<<<dim3((unsigned)(NN / 256), (unsigned)plan->n_views), 256, 0, st>>>(a);
    dm64::cols64_kernel<true><<<lines, N / 2, sm_cols, st>>>(a);
    dm64::rows64_kernel<false><<<lines, N / 2, sm_rows, st>>>(a);
    CU(cudaGetLastError());
    const int nO = 1 - plan->curO, nP = 1 - plan->curP;
    dm_status s = launch_object64(plan, st, plan->P64[plan->curP], plan->O64[plan->curO], plan->O64[nO], nullptr);
    if (s != DM_OK) return s;
    s = launch_probe64(plan, st, plan->O64[nO], plan->P64[plan->curP], plan->P64[nP], nullptr);
    if (s != DM_OK) return s;
    dm64::Err64 e;
    e.pF = plan->partF64; e.nF = (int)(plan->n_views * (NN / 256));
    e.pS = plan->partS64; e.nS = (int)lines;
    e.pP = plan->partP64; e.nP = (int)(NN / 256);
    e.pO = plan->partO64; e.nO = plan->nty * plan->ntx;
    e.K = plan->K; e.L = plan->L;
    e.row = plan->errors + (size_t)plan->rows * (2 + plan->K + plan->L);
    dm64::err64_finalize_kernel<<<2 + plan->K + plan->L, 1024, 0, st>>>(e);
    CU(cudaGetLastError());
    plan->curO = nO;
    plan->curP = nP;
    plan->rows++;
    return DM_OK;
}

// dm_set_data proper.  n_chunks > 0 (dm_solve_host): `intensities` arrives in n_chunks pieces of
// whole views, piece c being complete once chunk_ev[c] has fired; sqrt(I) is then formed piece by
// piece AFTER the kernels that do not need the data, so those run under the host-to-device copy.
dm_status set_data_impl(dm_plan *plan, const float *intensities, const float *probe0, const float *object0, void *stream,
                        const cudaEvent_t *chunk_ev, int n_chunks)
{
    dm_status s = check_ready(plan, false);
    if (s != DM_OK) return s;
    if (!intensities || !probe0 || !object0) return fail(plan, DM_ERR_INVALID_ARG, "NULL data pointer");
    int path = plan->path_req;
    if (path == 0) path = plan->N == 128 ? 3 : (plan->N < 128 ? 2 : 4);
    if (plan->precision == 1) path = 64;         // FP64 validation mode: its own plain kernels
    if (path == 2 && plan->N > 128)
        return fail(plan, DM_ERR_UNSUPPORTED, "fused per-frame path needs N <= 128 (N = %d)", plan->N);
    if (path == 3 && plan->N != 128)
        return fail(plan, DM_ERR_UNSUPPORTED, "register-resident path needs N = 128 (N = %d)", plan->N);
    plan->path = path;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t NN = (size_t)plan->N * plan->N, HW = (size_t)plan->H * plan->W;
    // spectrum layout of the chosen path (where sqrt(I) has to sit), twiddles and integer tables: uploaded once
    // per workspace and path (host-to-device copies of pageable memory would otherwise queue behind the
    // intensities of dm_solve_host on the copy engine)
    if (plan->tables_path != path) {
    plan->spec.assign(NN, 0);
    if (path == 3) {
        for (int tid = 0; tid < dmreg::RNT; ++tid)
            for (int e = 0; e < dmreg::REPT; ++e) plan->spec[dmreg::spec_pos(tid, e)] = dmreg::spec_freq(tid, e);
        std::vector<float> wy(256), wx(256);
        for (int w = 0; w < 16; ++w)
            for (int q = 0; q < 8; ++q) {
                const double ang = -2.0 * M_PI * (double)(w * q) / 128.0;
                wy[2 * (w * 8 + q)] = (float)std::cos(ang);
                wy[2 * (w * 8 + q) + 1] = (float)std::sin(ang);
            }
        for (int t = 0; t < 32; ++t)
            for (int r = 0; r < 4; ++r) {
                const double ang = -2.0 * M_PI * (double)(t * r) / 128.0;
                wx[2 * (t * 4 + r)] = (float)std::cos(ang);
                wx[2 * (t * 4 + r) + 1] = (float)std::sin(ang);
            }
        CU(cudaMemcpyAsync(plan->wy_d, wy.data(), 256 * sizeof(float), cudaMemcpyHostToDevice, st));
        CU(cudaMemcpyAsync(plan->wx_d, wx.data(), 256 * sizeof(float), cudaMemcpyHostToDevice, st));
        CU(cudaStreamSynchronize(st));          // wy / wx are stack-owned host buffers
    } else if (path == 4) {
        const int N = plan->N, RX = N / 32, G = 32 / RX;
        for (int cg = 0; cg < N / G; ++cg)
            for (int a = 0; a < 32; ++a)
                for (int k2 = 0; k2 < 32; ++k2) {
                    int f;
                    switch (N) {
                    case 64: f = dmwf::spec_freq<64>(cg, a, k2); break;
                    case 128: f = dmwf::spec_freq<128>(cg, a, k2); break;
                    case 256: f = dmwf::spec_freq<256>(cg, a, k2); break;
                    default: f = dmwf::spec_freq<512>(cg, a, k2); break;
                    }
                    plan->spec[dmwf::spec_pos(cg, a, k2)] = f;
                }
        std::vector<float> tw((size_t)RX * 32 * 2);
        for (int k1 = 0; k1 < RX; ++k1)
            for (int t = 0; t < 32; ++t) {
                const double ang = -2.0 * M_PI * (double)(t * k1) / (double)N;
                tw[2 * (k1 * 32 + t)] = (float)std::cos(ang);
                tw[2 * (k1 * 32 + t) + 1] = (float)std::sin(ang);
            }
        CU(cudaMemcpyAsync(plan->wf_tw_d, tw.data(), tw.size() * sizeof(float), cudaMemcpyHostToDevice, st));
        CU(cudaStreamSynchronize(st));          // tw is a stack-owned host buffer
    } else {
        for (int py = 0; py < plan->N; ++py)
            for (int px = 0; px < plan->N; ++px) plan->spec[(size_t)py * plan->N + px] = plan->rev[py] * plan->N + plan->rev[px];
    }
    CU(cudaMemcpyAsync(plan->pos_d, plan->pos.data(), plan->pos.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(plan->tile_ptr_d, plan->tile_ptr.data(), plan->tile_ptr.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    if (!plan->tile_views.empty())
        CU(cudaMemcpyAsync(plan->tile_views_d, plan->tile_views.data(), plan->tile_views.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(plan->spec_d, plan->spec.data(), plan->spec.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(plan->tw_d, plan->tw.data(), plan->tw.size() * sizeof(float), cudaMemcpyHostToDevice, st));
    CU(cudaStreamSynchronize(st));              // pageable host sources
    if (path != 64) {
        dm_status qs = launch_psi_update(plan, st, true);      // function attributes + occupancy-sized grids
        if (qs != DM_OK) return qs;
    }
    plan->tables_path = path;
    }
    if (plan->precision == 1) {
        for (int c = 0; c < n_chunks; ++c) CU(cudaStreamWaitEvent(st, chunk_ev[c], 0));
        s = set_data64(plan, intensities, probe0, object0, st);
        if (s != DM_OK) return s;
        plan->has_data = true;
        plan->rows = 0;
        return DM_OK;
    }
    plan->curP = plan->curO = 0;
    CU(cudaMemcpyAsync(plan->Pbuf[0], probe0, plan->K * NN * sizeof(float2), cudaMemcpyDeviceToDevice, st));
    CU(cudaMemcpyAsync(plan->Obuf[0], object0, plan->L * HW * sizeof(float2), cudaMemcpyDeviceToDevice, st));
    CU(cudaMemsetAsync(plan->alphas, 0, 2 * sizeof(float), st));
    const size_t total = (size_t)plan->n_views * NN;
    if (n_chunks <= 0) amp_permute_kernel<<<plan->sms * 8, 256, 0, st>>>(plan->N, intensities, plan->spec_d, plan->amp, total);
    psi_init_kernel<<<dim3((unsigned)((NN + 1023) / 1024), (unsigned)(plan->n_views * plan->M)), 256, 0, st>>>(
        plan->N, plan->K, plan->L, plan->H, plan->W, plan->pos_d, plan->Pbuf[0], plan->Obuf[0], plan->psi);
    CU(cudaGetLastError());
    // frozen regularisers (reading A8): alpha_O = a_O max_r den_O(P0), alpha_P = a_P max_r den_P(O0);
    // the two update kernels run once with alpha = 0 into the spare buffers just to produce den.
    s = launch_object(plan, st, plan->Pbuf[0], plan->Obuf[0], plan->Obuf[1], plan->den_tmp);
    if (s != DM_OK) return s;
    max_scale_kernel<<<1, 1024, 0, st>>>(plan->den_tmp, HW, (float)plan->a_obj, plan->alphas);
    s = launch_probe(plan, st, plan->Obuf[0], plan->Pbuf[0], plan->Pbuf[1], plan->den_tmp);
    if (s != DM_OK) return s;
    max_scale_kernel<<<1, 1024, 0, st>>>(plan->den_tmp, NN, (float)plan->a_probe, plan->alphas + 1);
    CU(cudaGetLastError());
    for (int c = 0; c < n_chunks; ++c) {
        const int v0 = (int)((long long)plan->n_views * c / n_chunks), v1 = (int)((long long)plan->n_views * (c + 1) / n_chunks);
        if (v1 == v0) continue;
        CU(cudaStreamWaitEvent(st, chunk_ev[c], 0));
        amp_permute_kernel<<<plan->sms * 8, 256, 0, st>>>(plan->N, intensities + (size_t)v0 * NN, plan->spec_d,
                                                    plan->amp + (size_t)v0 * NN, (size_t)(v1 - v0) * NN);
    }
    CU(cudaGetLastError());
    plan->has_data = true;
    plan->rows = 0;
    return DM_OK;
}
} // namespace

extern "C" {

dm_status dm_set_data(dm_plan *plan, const float *intensities, const float *probe0, const float *object0, void *stream)
{
    return set_data_impl(plan, intensities, probe0, object0, stream, nullptr, 0);
}

dm_status dm_iterate(dm_plan *plan, int n_iter, void *stream)
{
    dm_status s = check_ready(plan, true);
    if (s != DM_OK) return s;
    if (n_iter < 0) return fail(plan, DM_ERR_INVALID_ARG, "n_iter = %d < 0", n_iter);
    if (plan->rows + n_iter > ERR_ROWS_CAP)
        return fail(plan, DM_ERR_WORKSPACE, "error table holds %d rows; call dm_set_data to reset", ERR_ROWS_CAP);
    cudaStream_t st = (cudaStream_t)stream;
    const int ncol = 2 + plan->K + plan->L;
    for (int it = 0; it < n_iter && plan->precision == 1; ++it) {
        s = iterate64(plan, st);
        if (s != DM_OK) return s;
    }
    if (plan->precision == 1) return DM_OK;
    for (int it = 0; it < n_iter; ++it) {
        cudaEvent_t *ev = nullptr;
        if (plan->profiling && plan->ev_iters < PROF_MAX_ITERS) {
            while ((int)plan->ev.size() < 5 * (plan->ev_iters + 1)) {
                cudaEvent_t e;
                CU(cudaEventCreate(&e));
                plan->ev.push_back(e);
            }
            ev = plan->ev.data() + 5 * plan->ev_iters++;
        }
        if (ev) CU(cudaEventRecord(ev[0], st));
        s = launch_psi_update(plan, st);                                           // S1-S6
        if (s != DM_OK) return s;
        if (ev) CU(cudaEventRecord(ev[1], st));
        const int nO = 1 - plan->curO, nP = 1 - plan->curP;
        s = launch_object(plan, st, plan->Pbuf[plan->curP], plan->Obuf[plan->curO], plan->Obuf[nO], nullptr);   // S7
        if (s != DM_OK) return s;
        if (ev) CU(cudaEventRecord(ev[2], st));
        s = launch_probe(plan, st, plan->Obuf[nO], plan->Pbuf[plan->curP], plan->Pbuf[nP], nullptr);            // S8
        if (s != DM_OK) return s;
        if (ev) CU(cudaEventRecord(ev[3], st));
        ErrArgs e;                                                                   // S9
        if (plan->path == 4) {
            e.pF = plan->partA; e.nF = plan->n_views * plan->wf_nB; e.sF = 2;
            e.pS = plan->partB; e.nS = plan->n_views * plan->wf_nC; e.sS = 2;
        } else if (plan->path == 3) {
            e.pF = plan->partA;     e.nF = plan->reg_grid; e.sF = 4;
            e.pS = plan->partA + 2; e.nS = plan->reg_grid; e.sS = 4;
        } else if (plan->path == 2) {
            e.pF = plan->partA;     e.nF = plan->n_views * plan->M; e.sF = 4;
            e.pS = plan->partA + 2; e.nS = plan->n_views * plan->M; e.sS = 4;
        } else {
            e.pF = plan->partA; e.nF = plan->nA; e.sF = 2;
            e.pS = plan->partB; e.nS = plan->nB; e.sS = 2;
        }
        e.pP = plan->partP; e.nP = plan->fin_blocks;
        e.pO = plan->partO; e.nO = plan->nty * plan->ntx;
        e.K = plan->K; e.L = plan->L;
        e.row = plan->errors + (size_t)plan->rows * ncol;
        error_finalize_kernel<<<ncol, ERR_NT, 0, st>>>(e);
        CU(cudaGetLastError());
        if (ev) CU(cudaEventRecord(ev[4], st));
        plan->curO = nO;
        plan->curP = nP;
        plan->rows++;
    }
    return DM_OK;
}

dm_status dm_get_probe(const dm_plan *plan, float *out_dev, void *stream)
{
    dm_status s = check_ready(plan, true);
    if (s != DM_OK) return s;
    if (!out_dev) return fail(plan, DM_ERR_INVALID_ARG, "NULL output");
    if (plan->precision == 1) {
        dm64::d2f_kernel<<<CONV_GRID, 256, 0, (cudaStream_t)stream>>>((const double *)plan->P64[plan->curP], out_dev,
                                                                        2 * (size_t)plan->K * plan->N * plan->N);
        CU(cudaGetLastError());
        return DM_OK;
    }
    CU(cudaMemcpyAsync(out_dev, plan->Pbuf[plan->curP], (size_t)plan->K * plan->N * plan->N * sizeof(float2),
                       cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
    return DM_OK;
}

dm_status dm_get_object(const dm_plan *plan, float *out_dev, void *stream)
{
    dm_status s = check_ready(plan, true);
    if (s != DM_OK) return s;
    if (!out_dev) return fail(plan, DM_ERR_INVALID_ARG, "NULL output");
    if (plan->precision == 1) {
        dm64::d2f_kernel<<<CONV_GRID, 256, 0, (cudaStream_t)stream>>>((const double *)plan->O64[plan->curO], out_dev,
                                                                        2 * (size_t)plan->L * plan->H * plan->W);
        CU(cudaGetLastError());
        return DM_OK;
    }
    CU(cudaMemcpyAsync(out_dev, plan->Obuf[plan->curO], (size_t)plan->L * plan->H * plan->W * sizeof(float2),
                       cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
    return DM_OK;
}

dm_status dm_get_psi(const dm_plan *plan, float *out_dev, void *stream)
{
    dm_status s = check_ready(plan, true);
    if (s != DM_OK) return s;
    if (!out_dev) return fail(plan, DM_ERR_INVALID_ARG, "NULL output");
    if (plan->precision == 1) {
        dm64::d2f_kernel<<<CONV_GRID, 256, 0, (cudaStream_t)stream>>>((const double *)plan->psi64, out_dev,
                                                                        2 * (size_t)plan->n_views * plan->M * plan->N * plan->N);
        CU(cudaGetLastError());
        return DM_OK;
    }
    CU(cudaMemcpyAsync(out_dev, plan->psi, (size_t)plan->n_views * plan->M * plan->N * plan->N * sizeof(float2),
                       cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
    return DM_OK;
}

dm_status dm_get_errors(const dm_plan *plan, double *out_host, int max_rows, int *rows_written)
{
    dm_status s = check_ready(plan, true);
    if (s != DM_OK) return s;
    if (!out_host || !rows_written || max_rows < 0) return fail(plan, DM_ERR_INVALID_ARG, "bad output arguments");
    CU(cudaDeviceSynchronize());
    const int n = plan->rows < max_rows ? plan->rows : max_rows;
    if (n > 0) CU(cudaMemcpy(out_host, plan->errors, (size_t)n * (2 + plan->K + plan->L) * sizeof(double), cudaMemcpyDeviceToHost));
    *rows_written = n;
    return DM_OK;
}

dm_status dm_set_state(dm_plan *plan, const float *probe_dev, const float *object_dev, const float *psi_dev, void *stream)
{
    dm_status s = check_ready(plan, true);
    if (s != DM_OK) return s;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t NN = (size_t)plan->N * plan->N, HW = (size_t)plan->H * plan->W;
    if (plan->precision == 1) {
        if (probe_dev) dm64::f2d_kernel<<<CONV_GRID, 256, 0, st>>>(probe_dev, (double *)plan->P64[plan->curP], 2 * plan->K * NN, 0);
        if (object_dev) dm64::f2d_kernel<<<CONV_GRID, 256, 0, st>>>(object_dev, (double *)plan->O64[plan->curO], 2 * plan->L * HW, 0);
        if (psi_dev) dm64::f2d_kernel<<<CONV_GRID, 256, 0, st>>>(psi_dev, (double *)plan->psi64, 2 * (size_t)plan->n_views * plan->M * NN, 0);
        CU(cudaGetLastError());
        return DM_OK;
    }
    if (probe_dev) CU(cudaMemcpyAsync(plan->Pbuf[plan->curP], probe_dev, plan->K * NN * sizeof(float2), cudaMemcpyDeviceToDevice, st));
    if (object_dev) CU(cudaMemcpyAsync(plan->Obuf[plan->curO], object_dev, plan->L * HW * sizeof(float2), cudaMemcpyDeviceToDevice, st));
    if (psi_dev) CU(cudaMemcpyAsync(plan->psi, psi_dev, (size_t)plan->n_views * plan->M * NN * sizeof(float2), cudaMemcpyDeviceToDevice, st));
    return DM_OK;
}

dm_status dm_get_window_table(const dm_plan *plan, int32_t *out_host)
{
    if (!plan || !out_host) return DM_ERR_INVALID_ARG;
    for (int j = 0; j < plan->n_views; ++j) {
        out_host[3 * j] = plan->pos[2 * j];
        out_host[3 * j + 1] = plan->pos[2 * j + 1];
        out_host[3 * j + 2] = plan->pos[2 * j] * plan->W + plan->pos[2 * j + 1];
    }
    return DM_OK;
}

dm_status dm_get_coverage(const dm_plan *plan, int *tile_h, int *tile_w, int32_t *tile_ptr_host,
                          int32_t *tile_views_host, int64_t *nnz)
{
    if (!plan || !tile_h || !tile_w || !nnz) return DM_ERR_INVALID_ARG;
    *tile_h = OBJ_TH;
    *tile_w = OBJ_TW;
    *nnz = (int64_t)plan->tile_views.size();
    if (tile_ptr_host) memcpy(tile_ptr_host, plan->tile_ptr.data(), plan->tile_ptr.size() * sizeof(int32_t));
    if (tile_views_host && !plan->tile_views.empty())
        memcpy(tile_views_host, plan->tile_views.data(), plan->tile_views.size() * sizeof(int32_t));
    return DM_OK;
}

dm_status dm_get_alphas(const dm_plan *plan, double *out_host2)
{
    dm_status s = check_ready(plan, true);
    if (s != DM_OK) return s;
    if (!out_host2) return fail(plan, DM_ERR_INVALID_ARG, "NULL output");
    CU(cudaDeviceSynchronize());
    if (plan->precision == 1) {
        CU(cudaMemcpy(out_host2, plan->alphas64, 2 * sizeof(double), cudaMemcpyDeviceToHost));
        return DM_OK;
    }
    float a[2];
    CU(cudaMemcpy(a, plan->alphas, sizeof a, cudaMemcpyDeviceToHost));
    out_host2[0] = a[0];
    out_host2[1] = a[1];
    return DM_OK;
}

dm_status dm_get_mode_power(const dm_plan *plan, double *out_host)
{
    dm_status s = check_ready(plan, true);
    if (s != DM_OK) return s;
    if (!out_host) return fail(plan, DM_ERR_INVALID_ARG, "NULL output");
    const size_t NN = (size_t)plan->N * plan->N, HW = (size_t)plan->H * plan->W;
    CU(cudaDeviceSynchronize());
    if (plan->precision == 1) {     // the FP32 state buffers are unused in this mode: park the rounded state there
        dm64::d2f_kernel<<<CONV_GRID, 256>>>((const double *)plan->P64[plan->curP], (float *)plan->Pbuf[plan->curP], 2 * plan->K * NN);
        dm64::d2f_kernel<<<CONV_GRID, 256>>>((const double *)plan->O64[plan->curO], (float *)plan->Obuf[plan->curO], 2 * plan->L * HW);
    }
    mode_power_kernel<<<plan->K, 1024>>>(plan->Pbuf[plan->curP], NN, plan->mode_pow);
    mode_power_kernel<<<plan->L, 1024>>>(plan->Obuf[plan->curO], HW, plan->mode_pow + plan->K);
    CU(cudaGetLastError());
    CU(cudaMemcpy(out_host, plan->mode_pow, (size_t)(plan->K + plan->L) * sizeof(double), cudaMemcpyDeviceToHost));
    double tp = 0.0, to = 0.0;
    for (int k = 0; k < plan->K; ++k) tp += out_host[k];
    for (int l = 0; l < plan->L; ++l) to += out_host[plan->K + l];
    for (int k = 0; k < plan->K; ++k) out_host[k] = tp > 0.0 ? out_host[k] / tp : 0.0;
    for (int l = 0; l < plan->L; ++l) out_host[plan->K + l] = to > 0.0 ? out_host[plan->K + l] / to : 0.0;
    return DM_OK;
}

dm_status dm_solve_host(dm_plan *plan, const float *intensities_host, const float *probe0_host,
                        const float *object0_host, int n_iter, float *out_probe_host, float *out_object_host,
                        void *stream)
{
    dm_status s = check_ready(plan, false);
    if (s != DM_OK) return s;
    if (!intensities_host || !probe0_host || !object0_host) return fail(plan, DM_ERR_INVALID_ARG, "NULL data pointer");
    cudaStream_t st = (cudaStream_t)stream;
    const size_t NN = (size_t)plan->N * plan->N, HW = (size_t)plan->H * plan->W;
    constexpr int NCH = 8;
    if (!plan->copy_ready) {
        CU(cudaStreamCreateWithFlags(&plan->copy_st, cudaStreamNonBlocking));
        CU(cudaEventCreateWithFlags(&plan->ev_begin, cudaEventDisableTiming));
        for (int c = 0; c < NCH; ++c) CU(cudaEventCreateWithFlags(&plan->ev_chunk[c], cudaEventDisableTiming));
        plan->copy_ready = true;
    }
    // P0, O0 (small) first on the caller's stream; the intensities in NCH chunks on the copy stream,
    // which starts once everything already queued on `st` (earlier readers of the staging area) is done
    CU(cudaEventRecord(plan->ev_begin, st));
    CU(cudaStreamWaitEvent(plan->copy_st, plan->ev_begin, 0));
    CU(cudaMemcpyAsync(plan->stage_P, probe0_host, plan->K * NN * sizeof(float2), cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(plan->stage_O, object0_host, plan->L * HW * sizeof(float2), cudaMemcpyHostToDevice, st));
    for (int c = 0; c < NCH; ++c) {
        const size_t v0 = (size_t)((long long)plan->n_views * c / NCH), v1 = (size_t)((long long)plan->n_views * (c + 1) / NCH);
        if (v1 > v0)
            CU(cudaMemcpyAsync(plan->stage_I + v0 * NN, intensities_host + v0 * NN, (v1 - v0) * NN * sizeof(float),
                               cudaMemcpyHostToDevice, plan->copy_st));
        CU(cudaEventRecord(plan->ev_chunk[c], plan->copy_st));
    }
    plan->has_data = false;
    s = set_data_impl(plan, plan->stage_I, (const float *)plan->stage_P, (const float *)plan->stage_O, stream, plan->ev_chunk, NCH);
    if (s != DM_OK) return s;
    s = dm_iterate(plan, n_iter, stream);
    if (s != DM_OK) return s;
    if (plan->precision == 1) {     // round the FP64 state into the FP32 state buffers (unused in this mode)
        dm64::d2f_kernel<<<CONV_GRID, 256, 0, st>>>((const double *)plan->P64[plan->curP], (float *)plan->Pbuf[plan->curP], 2 * plan->K * NN);
        dm64::d2f_kernel<<<CONV_GRID, 256, 0, st>>>((const double *)plan->O64[plan->curO], (float *)plan->Obuf[plan->curO], 2 * plan->L * HW);
    }
    if (out_probe_host)
        CU(cudaMemcpyAsync(out_probe_host, plan->Pbuf[plan->curP], plan->K * NN * sizeof(float2), cudaMemcpyDeviceToHost, st));
    if (out_object_host)
        CU(cudaMemcpyAsync(out_object_host, plan->Obuf[plan->curO], plan->L * HW * sizeof(float2), cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    return DM_OK;
}

dm_status dm_plan_set_profiling(dm_plan *plan, int on)
{
    if (!plan) return DM_ERR_INVALID_ARG;
    plan->profiling = on != 0;
    plan->ev_iters = 0;
    return DM_OK;
}

dm_status dm_get_phase_ms(dm_plan *plan, float *out_ms4, int *iters)
{
    if (!plan || !out_ms4 || !iters) return DM_ERR_INVALID_ARG;
    CU(cudaDeviceSynchronize());
    double acc[4] = {0, 0, 0, 0};
    for (int i = 0; i < plan->ev_iters; ++i)
        for (int ph = 0; ph < 4; ++ph) {
            float ms = 0.f;
            CU(cudaEventElapsedTime(&ms, plan->ev[5 * i + ph], plan->ev[5 * i + ph + 1]));
            acc[ph] += ms;
        }
    for (int ph = 0; ph < 4; ++ph) out_ms4[ph] = (float)acc[ph];
    *iters = plan->ev_iters;
    plan->ev_iters = 0;
    return DM_OK;
}

dm_status dm_plan_info(const dm_plan *plan, int *path, int *launches_per_iter)
{
    if (!plan) return DM_ERR_INVALID_ARG;
    int p = plan->path ? plan->path : (plan->path_req ? plan->path_req : (plan->N == 128 ? 3 : (plan->N < 128 ? 2 : 4)));
    if (plan->precision == 1) p = 64;
    if (path) *path = p;
    if (launches_per_iter) {
        const int chunks = (plan->n_views + plan->chunk_views - 1) / plan->chunk_views;
        *launches_per_iter = p == 64 ? 8 : (p >= 2 ? 1 : 3 * chunks) + 4;
    }
    return DM_OK;
}

dm_status dm_plan_geometry(const dm_plan *plan, int32_t *out_host, int n_out)
{
    if (!plan || !out_host || n_out < 0) return DM_ERR_INVALID_ARG;
    int path = 0;
    dm_plan_info(plan, &path, nullptr);
    const bool reg = path == 3;
    const int per_view = plan->M;
    const int clusters = reg && plan->reg_grid > 0 ? plan->reg_grid / per_view : 0;
    const int32_t g[DM_GEOMETRY_FIELDS] = {
        path, plan->sms, plan->prb_chunks, plan->prb_chunk_len, plan->max_list, OBJ_NT,
        reg ? plan->reg_grid : 0, reg ? per_view : 0, clusters ? (plan->n_views + clusters - 1) / clusters : 0,
        plan->wf_S, plan->wf_D, path == 4 ? plan->wf_grid : 0, plan->wf_nw, reg && plan->reg_sw ? 1 : 0};
    for (int i = 0; i < n_out && i < DM_GEOMETRY_FIELDS; ++i) out_host[i] = g[i];
    return DM_OK;
}

} // extern "C"

namespace {
struct NoSync { __host__ __device__ void operator()() const {} };
template <int N> void host_fft2(const float *in, float *out, int inverse)
{
    std::vector<float2> tile((size_t)N * N), tw(N);
    for (int n = 0; n < N; ++n) {
        const double ang = -2.0 * M_PI * (double)n / (double)N;
        tw[n] = make_float2((float)std::cos(ang), (float)std::sin(ang));
    }
    std::vector<int32_t> rev;
    fill_rev<N>(rev);
    const float2 *src = reinterpret_cast<const float2 *>(in);
    float2 *dst = reinterpret_cast<float2 *>(out);
    if (!inverse) {
        for (int e = 0; e < N * N; ++e) tile[swz(e)] = src[e];
        // emulate NT threads one after the other: butterflies of one pass touch disjoint elements
        for (int t = 0; t < 64; ++t) tile_pass<N, Radix<N>::R1, N, false, false, N, N>(tile.data(), tw.data(), t, 64);
        for (int t = 0; t < 64; ++t) tile_pass<N, Radix<N>::R2, N / Radix<N>::R1, false, false, N, N>(tile.data(), tw.data(), t, 64);
        if (Radix<N>::R3 > 1)
            for (int t = 0; t < 64; ++t) tile_pass<N, (Radix<N>::R3 > 1 ? Radix<N>::R3 : 2), (Radix<N>::R3 > 1 ? N / (Radix<N>::R1 * Radix<N>::R2) : 2), false, false, N, N>(tile.data(), tw.data(), t, 64);
        axis_fft<N, false, true, N, N>(tile.data(), tw.data(), 0, 1, NoSync());
        for (int py = 0; py < N; ++py)
            for (int px = 0; px < N; ++px) dst[(size_t)rev[py] * N + rev[px]] = tile[swz(py * N + px)];
    } else {
        // input is a natural-order spectrum: place it in the kernels' permuted layout first
        for (int py = 0; py < N; ++py)
            for (int px = 0; px < N; ++px) tile[swz(py * N + px)] = src[(size_t)rev[py] * N + rev[px]];
        axis_fft<N, true, true, N, N>(tile.data(), tw.data(), 0, 1, NoSync());
        axis_fft<N, true, false, N, N>(tile.data(), tw.data(), 0, 1, NoSync());
        const float s = 1.f / ((float)N * (float)N);
        for (int e = 0; e < N * N; ++e) dst[e] = make_float2(tile[swz(e)].x * s, tile[swz(e)].y * s);
    }
}
// path 3 (dm_regfft.cuh): 512 emulated threads, phase by phase (a phase boundary = a barrier)
void host_fft2_reg(const float *in, float *out, int inverse)
{
    using namespace dmreg;
    std::vector<float2> regs((size_t)RNT * REPT);
    std::vector<float4> xbuf_v(XBUF3_BYTES / 16);      // the kernel's exchange buffer: 64 KiB + the 16 spare strips
    unsigned char *xbuf = reinterpret_cast<unsigned char *>(xbuf_v.data());
    std::vector<float2> wy(128), wx(128);
    for (int w = 0; w < 16; ++w)
        for (int q = 0; q < 8; ++q) {
            const double ang = -2.0 * M_PI * (double)(w * q) / 128.0;
            wy[w * 8 + q] = make_float2((float)std::cos(ang), (float)std::sin(ang));
        }
    for (int t = 0; t < 32; ++t)
        for (int r = 0; r < 4; ++r) {
            const double ang = -2.0 * M_PI * (double)(t * r) / 128.0;
            wx[t * 4 + r] = make_float2((float)std::cos(ang), (float)std::sin(ang));
        }
    auto U = [&](int tid) -> float2(&)[32] { return *reinterpret_cast<float2(*)[32]>(&regs[(size_t)tid * REPT]); };
    const float2 *src = reinterpret_cast<const float2 *>(in);
    float2 *dst = reinterpret_cast<float2 *>(out);
    auto exch1 = [&]() {
        for (int rho = 0; rho < 2; ++rho) {
            // the kernel's own addressing: a warp's rows 0..27 inside its 4 KiB exchange-2 region, rows 28..31 in its spare strip
            for (int tid = 0; tid < RNT; ++tid)
                x1s_write(U(tid), rho, tid & 31, xbuf + (tid >> 5) * 4096, xbuf + X1S_SPARE_OFF + (tid >> 5) * X1S_SPARE);
            for (int tid = 0; tid < RNT; ++tid)
                x1s_read(U(tid), rho, tid & 31, xbuf + (tid >> 5) * 4096, xbuf + X1S_SPARE_OFF + (tid >> 5) * X1S_SPARE);
        }
    };
    auto exch2 = [&]() {
        for (int z = 0; z < 2; ++z) {
            for (int tid = 0; tid < RNT; ++tid) x2_write(U(tid), z, tid >> 5, tid & 31, reinterpret_cast<float2 *>(xbuf));
            for (int tid = 0; tid < RNT; ++tid) x2_read(U(tid), z, tid >> 5, tid & 31, reinterpret_cast<const float2 *>(xbuf));
        }
    };
    if (!inverse) {
        for (int tid = 0; tid < RNT; ++tid)
            for (int a = 0; a < REPT; ++a) U(tid)[a] = src[l0_pixel(tid, a)];
        for (int tid = 0; tid < RNT; ++tid) pass1_fwd(U(tid), &wy[(tid >> 5) * 8], &wx[(tid & 31) * 4]);
        exch1();
        for (int tid = 0; tid < RNT; ++tid) pass2<false>(U(tid));
        exch2();
        for (int tid = 0; tid < RNT; ++tid) pass3<false>(U(tid));
        for (int tid = 0; tid < RNT; ++tid)
            for (int e = 0; e < REPT; ++e) dst[spec_freq(tid, e)] = U(tid)[e];
    } else {
        for (int tid = 0; tid < RNT; ++tid)
            for (int e = 0; e < REPT; ++e) U(tid)[e] = src[spec_freq(tid, e)];
        for (int tid = 0; tid < RNT; ++tid) pass3<true>(U(tid));
        exch2();
        for (int tid = 0; tid < RNT; ++tid) pass2<true>(U(tid));
        exch1();
        for (int tid = 0; tid < RNT; ++tid) pass1_inv(U(tid), &wy[(tid >> 5) * 8], &wx[(tid & 31) * 4]);
        const float s = 1.f / (float)RNN;
        for (int tid = 0; tid < RNT; ++tid)
            for (int a = 0; a < REPT; ++a) dst[l0_pixel(tid, a)] = make_float2(U(tid)[a].x * s, U(tid)[a].y * s);
    }
}
// path 4 (dm_warpfft.cuh): one emulated warp (32 lanes, phase by phase) per row group / column group
template <int N> void host_fft2_wf(const float *in, float *out, int inverse)
{
    using namespace dmwf;
    constexpr int RX = N / 32, G = 32 / RX, NG = N / G;
    std::vector<float2> tw((size_t)RX * 32), scratch((size_t)N * N), regs(32 * 32);
    std::vector<float4> xbuf_v(WF_XBUF / 16);
    unsigned char *xbuf = reinterpret_cast<unsigned char *>(xbuf_v.data());
    for (int k1 = 0; k1 < RX; ++k1)
        for (int t = 0; t < 32; ++t) {
            const double ang = -2.0 * M_PI * (double)(t * k1) / (double)N;
            tw[k1 * 32 + t] = make_float2((float)std::cos(ang), (float)std::sin(ang));
        }
    auto U = [&](int lane) -> float2(&)[32] { return *reinterpret_cast<float2(*)[32]>(&regs[(size_t)lane * 32]); };
    auto exch = [&]() {
        for (int t = 0; t < 32; ++t) xt_write(U(t), t, xbuf);
        for (int t = 0; t < 32; ++t) xt_read(U(t), t, xbuf);
    };
    auto fwd = [&]() {
        for (int t = 0; t < 32; ++t) stage1_fwd<RX>(U(t), tw.data(), t);
        exch();
        for (int t = 0; t < 32; ++t) dmreg::dft32<false>(U(t));
    };
    auto inv = [&]() {
        for (int t = 0; t < 32; ++t) dmreg::dft32<true>(U(t));
        exch();
        for (int t = 0; t < 32; ++t) stage1_inv<RX>(U(t), tw.data(), t);
    };
    const float2 *src = reinterpret_cast<const float2 *>(in);
    float2 *dst = reinterpret_cast<float2 *>(out);
    if (!inverse) {
        for (int rg = 0; rg < NG; ++rg) {                      // phase A: rows
            for (int t = 0; t < 32; ++t)
                for (int i = 0; i < 32; ++i) U(t)[i] = src[(size_t)(rg * G + i / RX) * N + t + 32 * (i % RX)];
            fwd();
            for (int a = 0; a < 32; ++a)
                for (int k2 = 0; k2 < 32; ++k2) scratch[scratch_index<N>(rg * G + a / RX, a % RX + RX * k2)] = U(a)[k2];
        }
        for (int cg = 0; cg < NG; ++cg) {                      // phase B: columns
            for (int t = 0; t < 32; ++t)
                for (int i = 0; i < 32; ++i) U(t)[i] = scratch[((size_t)cg * N + t + 32 * (i % RX)) * G + i / RX];
            fwd();
            for (int a = 0; a < 32; ++a)
                for (int k2 = 0; k2 < 32; ++k2) dst[spec_freq<N>(cg, a, k2)] = U(a)[k2];
        }
    } else {
        for (int cg = 0; cg < NG; ++cg) {
            for (int a = 0; a < 32; ++a)
                for (int k2 = 0; k2 < 32; ++k2) U(a)[k2] = src[spec_freq<N>(cg, a, k2)];
            inv();
            for (int t = 0; t < 32; ++t)
                for (int i = 0; i < 32; ++i) scratch[((size_t)cg * N + t + 32 * (i % RX)) * G + i / RX] = U(t)[i];
        }
        const float sc = 1.f / ((float)N * (float)N);
        for (int rg = 0; rg < NG; ++rg) {
            for (int a = 0; a < 32; ++a)
                for (int k2 = 0; k2 < 32; ++k2) U(a)[k2] = scratch[scratch_index<N>(rg * G + a / RX, a % RX + RX * k2)];
            inv();
            for (int t = 0; t < 32; ++t)
                for (int i = 0; i < 32; ++i) {
                    const float2 v = U(t)[i];
                    dst[(size_t)(rg * G + i / RX) * N + t + 32 * (i % RX)] = make_float2(v.x * sc, v.y * sc);
                }
        }
    }
}
} // namespace

extern "C" {

dm_status dm_host_fft2_path(int N, int path, const float *in_host, float *out_host, int inverse)
{
    if (!in_host || !out_host) return DM_ERR_INVALID_ARG;
    if (path == 3) {
        if (N != 128) return DM_ERR_UNSUPPORTED;
        host_fft2_reg(in_host, out_host, inverse);
        return DM_OK;
    }
    if (path == 4) {
        switch (N) {
        case 64: host_fft2_wf<64>(in_host, out_host, inverse); break;
        case 128: host_fft2_wf<128>(in_host, out_host, inverse); break;
        case 256: host_fft2_wf<256>(in_host, out_host, inverse); break;
        case 512: host_fft2_wf<512>(in_host, out_host, inverse); break;
        default: return DM_ERR_UNSUPPORTED;
        }
        return DM_OK;
    }
    if (path != 1 && path != 2) return DM_ERR_INVALID_ARG;
    return dm_host_fft2(N, in_host, out_host, inverse);
}

dm_status dm_host_fft2(int N, const float *in_host, float *out_host, int inverse)
{
    if (!in_host || !out_host) return DM_ERR_INVALID_ARG;
    switch (N) {
    case 64: host_fft2<64>(in_host, out_host, inverse); break;
    case 128: host_fft2<128>(in_host, out_host, inverse); break;
    case 256: host_fft2<256>(in_host, out_host, inverse); break;
    case 512: host_fft2<512>(in_host, out_host, inverse); break;
    default: return DM_ERR_UNSUPPORTED;
    }
    return DM_OK;
}

const char *dm_status_string(dm_status s)
{
    switch (s) {
    case DM_OK: return "DM_OK";
    case DM_ERR_INVALID_ARG: return "DM_ERR_INVALID_ARG";
    case DM_ERR_OUT_OF_BOUNDS: return "DM_ERR_OUT_OF_BOUNDS";
    case DM_ERR_UNSUPPORTED: return "DM_ERR_UNSUPPORTED";
    case DM_ERR_NO_DATA: return "DM_ERR_NO_DATA";
    case DM_ERR_WORKSPACE: return "DM_ERR_WORKSPACE";
    case DM_ERR_CUDA: return "DM_ERR_CUDA";
    }
    return "DM_ERR_?";
}

const char *dm_last_error(const dm_plan *plan) { return plan ? plan->err.c_str() : g_create_error.c_str(); }

void dm_plan_destroy(dm_plan *plan)
{
    if (!plan) return;
    for (cudaEvent_t e : plan->ev) cudaEventDestroy(e);
    if (plan->copy_ready) {
        cudaStreamDestroy(plan->copy_st);
        cudaEventDestroy(plan->ev_begin);
        for (int c = 0; c < 8; ++c) cudaEventDestroy(plan->ev_chunk[c]);
    }
    delete plan;
}

} // extern "C"
