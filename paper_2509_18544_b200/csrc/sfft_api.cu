// sfft_api.cu -- the C ABI of include/sfft.h: plan life cycle, stage sequencing, introspection.
// Every compute step is a kernel of this library (sfft_fwd/lags/assemble/solve/subtract.cu);
// this file only validates, allocates, orders launches on the plan's stream and times them.
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <cmath>
#include <new>
#include "sfft_internal.h"

using namespace sfft;

namespace sfft {

__global__ void twiddle_kernel(cplx *tw, int Nt) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= Nt) return;
    double s, c;
    sincospi(-2.0 * (double)k / (double)Nt, &s, &c);
    tw[k] = mk(c, s);
}

static void poly_index(int t, int *i, int *j) { // total degree ascending, then j ascending (reading C4)
    int d = 0;
    while (t > d) { t -= d + 1; d++; }
    *j = t; *i = d - t;
}

static int next_pow2(int v, int lo) { int m = lo; while (m < v) m <<= 1; return m; }

// sum_x xt(x)^k, xt = (2x+1-n)/n: exactly 0 for odd k (pin P7), long double otherwise
static double power_sum(int n, int k) {
    if (k & 1) return 0.0;
    long double acc = 0.0L;
    for (int x = 0; x < n; x++) {
        long double t = (2.0L * x + 1.0L - n) / n, p = 1.0L;
        for (int e = 0; e < k; e++) p *= t;
        acc += p;
    }
    return (double)acc;
}

} // namespace sfft

static sfft_status fail(sfft_plan *p, sfft_status st, const char *what, cudaError_t e = cudaSuccess) {
    if (p) {
        if (e != cudaSuccess) snprintf(p->err, sizeof(p->err), "%s: %s", what, cudaGetErrorString(e));
        else snprintf(p->err, sizeof(p->err), "%s", what);
    }
    return st;
}

#define CK(call, what)                                                          \
    do {                                                                        \
        cudaError_t e_ = (call);                                                \
        if (e_ != cudaSuccess) return fail(p, SFFT_ERR_CUDA, what, e_);         \
    } while (0)

template <typename T> static cudaError_t dalloc(sfft_plan *p, T **ptr, size_t count) {
    cudaError_t e = cudaMalloc((void **)ptr, count * sizeof(T));
    if (e == cudaSuccess) p->bytes += count * sizeof(T);
    return e;
}

struct StageTimer {
    sfft_plan *p; int stage;
    StageTimer(sfft_plan *p_, int s) : p(p_), stage(s) {
        if (p->timing) { cudaEventRecord(p->ev0[stage], p->cur); p->ev_used[stage] = true; }
    }
    ~StageTimer() { if (p->timing) cudaEventRecord(p->ev1[stage], p->cur); }
};

static void free_plan(sfft_plan *p) {
    if (!p) return;
    void *ptrs[] = {p->tw, p->inter, p->specT, (p->specTo != p->specT) ? p->specTo : nullptr, p->specS, p->muR, p->muS,
                    p->Q, p->phO, p->phT, p->lagO, p->lagT, p->bpart, p->SB, p->LP, p->gamA, p->gam, p->gamP, p->phi, p->delta, p->G, p->h, p->Lf, p->dscale, p->Linv,
                    p->ywork, p->zwork, p->coef, p->ratioEZ, p->ratioW, p->E, p->wcorr, p->flag, p->stS, p->stR, p->stD, p->stM};
    for (void *q : ptrs) if (q) cudaFree(q);
    for (int i = 1; i < NSCI; i++) { if (p->specSx[i]) cudaFree(p->specSx[i]); if (p->muSx[i]) cudaFree(p->muSx[i]); if (p->deltax[i]) cudaFree(p->deltax[i]); }
    for (int i = 1; i < 2 * NSCI; i++) { if (p->hq[i]) cudaFree(p->hq[i]); if (p->cq[i]) cudaFree(p->cq[i]); }
    if (p->flag_host) cudaFreeHost(p->flag_host);
    if (p->gmeta) cudaFree(p->gmeta);
    lags_free(p); rows_free(p);
    for (int s = 0; s < SFFT_NUM_STAGES; s++) {
        if (p->ev0[s]) cudaEventDestroy(p->ev0[s]);
        if (p->ev1[s]) cudaEventDestroy(p->ev1[s]);
    }
    if (p->side) cudaStreamDestroy(p->side);
    if (p->sideB) cudaStreamDestroy(p->sideB);
    if (p->sideC) cudaStreamDestroy(p->sideC);
    if (p->ev_joinB) cudaEventDestroy(p->ev_joinB);
    if (p->ev_joinC) cudaEventDestroy(p->ev_joinC);
    if (p->ev_fork) cudaEventDestroy(p->ev_fork);
    if (p->ev_join) cudaEventDestroy(p->ev_join);
    if (p->fstream) cudaStreamDestroy(p->fstream);
    if (p->ev_ffork) cudaEventDestroy(p->ev_ffork);
    if (p->cstream) cudaStreamDestroy(p->cstream);
    if (p->ostream) cudaStreamDestroy(p->ostream);
    for (int k = 0; k < 3; k++) {
        if (p->hbS[k]) cudaFree(p->hbS[k]); if (p->hbD[k]) cudaFree(p->hbD[k]); if (p->hbC[k]) cudaFree(p->hbC[k]);
        if (p->ev_hin[k]) cudaEventDestroy(p->ev_hin[k]); if (p->ev_hcomp[k]) cudaEventDestroy(p->ev_hcomp[k]); if (p->ev_hout[k]) cudaEventDestroy(p->ev_hout[k]);
    }
    if (p->ev_copy) cudaEventDestroy(p->ev_copy);
    if (p->ev_fjoin) cudaEventDestroy(p->ev_fjoin);
    if (p->fstream2) cudaStreamDestroy(p->fstream2);
    for (int k = 0; k < MAX_NP - 2; k++) { if (p->rstream[k]) cudaStreamDestroy(p->rstream[k]); if (p->ev_rjoin[k]) cudaEventDestroy(p->ev_rjoin[k]); }
    if (p->ev_rfork) cudaEventDestroy(p->ev_rfork);
    if (p->ev_lookP) cudaEventDestroy(p->ev_lookP);
    if (p->ev_lookB) cudaEventDestroy(p->ev_lookB);
    for (int k = 0; k < MAX_KREC; k++)
        if (p->krec[k].e0) { cudaEventDestroy(p->krec[k].e0); cudaEventDestroy(p->krec[k].e1); }
    delete p;
}

extern "C" {

const char *sfft_version(void) { return "sfft-b200 0.1 (sm_100a)"; }

sfft_status sfft_plan_create(sfft_plan **out, int nx, int ny, int L, int DK, int DB) {
    return sfft_plan_create_ex(out, nx, ny, L, DK, DB, 0u);
}

sfft_status sfft_plan_create_ex(sfft_plan **out, int nx, int ny, int L, int DK, int DB, unsigned flags) {
    if (!out) return SFFT_ERR_INVALID_ARG;
    if (flags & ~(unsigned)SFFT_PLAN_FP32_SPECTRA) return SFFT_ERR_INVALID_ARG;
    *out = nullptr;
    if (L < 1 || L > MAX_L || !(L & 1) || DK < 0 || DK > MAX_DEG || DB < 0 || DB > MAX_DEG) return SFFT_ERR_INVALID_ARG;
    if (nx < 2 * L - 1 || ny < 2 * L - 1 || nx > SFFT_MAX_SIDE || ny > SFFT_MAX_SIDE) return SFFT_ERR_INVALID_ARG;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); return SFFT_ERR_CUDA; }
    sfft_plan *p = new (std::nothrow) sfft_plan();
    if (!p) return SFFT_ERR_ALLOC;
    memset(p, 0, sizeof(*p));
    p->spec32 = (flags & SFFT_PLAN_FP32_SPECTRA) != 0; p->spec_esz = p->spec32 ? 8 : 16;
    Geom &g = p->g;
    g.nx = nx; g.ny = ny; g.L = L; g.w = (L - 1) / 2; g.DK = DK; g.DB = DB;
    g.NK = (DK + 1) * (DK + 2) / 2; g.NB = (DB + 1) * (DB + 2) / 2; g.n = L * L * g.NK + g.NB;
    // zero-padded FFT grid: powers of two, at least 1024 x 512 (the transforms run 16 values per thread in groups of
    // at least one warp; a small frame only pays a few MB of padding, the wrap corrections make any padding exact)
    g.Mx = next_pow2(nx, 1024); g.My = next_pow2(ny, 512); g.Hx = g.Mx / 2;
    g.log2Hx = ilog2(g.Hx); g.log2My = ilog2(g.My);
    g.Nt = g.Mx > g.My ? g.Mx : g.My;
    for (int t = 0; t < MAX_NP; t++) poly_index(t, &g.pi[t], &g.pj[t]);
    // pair lists: Omega t <= t' ; Theta (t, science)
    p->plO.np = 0;
    for (int t = 0; t < g.NK; t++)
        for (int tp = t; tp < g.NK; tp++) { p->plO.a[p->plO.np] = t; p->plO.b[p->plO.np] = tp; p->plO.np++; }
    p->plT.np = g.NK;
    for (int q = 0; q < MAX_PAIRS; q++) p->plT.ord[q] = q;
    for (int t = 0; t < g.NK; t++) { p->plT.a[t] = t; p->plT.b[t] = g.NK; }
    p->npairsO = p->plO.np;
    {   // slot order of the Omega pass: the NK self-pairs first
        int k = 0;
        for (int q = 0; q < p->plO.np; q++) if (p->plO.a[q] == p->plO.b[q]) p->plO.ord[k++] = q;
        for (int q = 0; q < p->plO.np; q++) if (p->plO.a[q] != p->plO.b[q]) p->plO.ord[k++] = q;
    }

    const size_t iplane = (size_t)g.My * g.Hx, splane = (size_t)g.My * (g.Hx + 1);
    const int W2 = 4 * g.w + 1, n = g.n;
    {   // experiment knobs: the environment is read here and nowhere else
        Knobs &k = p->knob;
        k.no_side = getenv("SFFT_NO_SIDE") != nullptr;
        k.no_factor_overlap = getenv("SFFT_NO_FACTOR_OVERLAP") != nullptr;
        k.no_batch_pipe = getenv("SFFT_NO_BATCH_PIPE") != nullptr;
        k.no_lookahead = getenv("SFFT_NO_LOOKAHEAD") != nullptr;
        const char *e = getenv("SFFT_BATCH_GROUP"); k.batch_group = e ? atoi(e) : NSCI;
        if (k.batch_group < 1 || k.batch_group > NSCI) k.batch_group = NSCI;
        e = getenv("SFFT_FACTOR_SMS"); k.factor_sms = e ? atoi(e) : 12;
        int dev = 0; cudaGetDevice(&dev);
        if (cudaDeviceGetAttribute(&p->sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || p->sms <= 0) p->sms = 148;
    }
    // lag-pass launch shapes first: they size Q
    lagcol_config(g, p->plO.np, g.NK, 2 * g.w, &p->cfgO, p->spec_esz);
    for (int k = 1; k <= NSCI; k++) lagcol_config(g, k * g.NK, g.NK + k, g.w, &p->cfgT[k - 1], p->spec_esz);
    size_t bO = (size_t)border_chunks() * p->plO.np * W2 * W2;
    { const size_t bT2 = (size_t)border_chunks() * NSCI * g.NK * L * L; if (bT2 > bO) bO = bT2; }
    cudaError_t e = cudaSuccess;
#define AL(ptr, cnt) if (e == cudaSuccess) e = dalloc(p, &ptr, (size_t)(cnt))
    AL(p->tw, g.Nt);
    AL(p->inter, (size_t)(DK + 1) * iplane);
#define ALB(ptr_, nb_) if (e == cudaSuccess) { e = cudaMalloc(&ptr_, (size_t)(nb_)); if (e == cudaSuccess) p->bytes += (size_t)(nb_); }
    ALB(p->specT, g.NK * splane * p->spec_esz);
    ALB(p->specS, splane * p->spec_esz);
    p->specSx[0] = p->specS;
    for (int i = 1; i < NSCI; i++) ALB(p->specSx[i], splane * p->spec_esz); // batched path: up to NSCI science spectra per Theta pass
#undef ALB
    AL(p->muR, (size_t)(DK + DB + 1) * ny);
    AL(p->muS, (size_t)(DB + 1) * ny);
    for (int i = 1; i < NSCI; i++) AL(p->muSx[i], (size_t)(DB + 1) * ny);
    AL(p->Q, lag_q_elems(p));
    AL(p->phO, (size_t)(g.My / 16) * p->cfgO.WB);
    AL(p->phT, (size_t)(g.My / 16) * p->cfgT[0].WB);
    AL(p->lagO, (size_t)p->plO.np * W2 * W2);
    AL(p->lagT, (size_t)NSCI * g.NK * L * L);
    AL(p->bpart, bO);
    AL(p->SB, border_strip_doubles(g, 2 * g.w > 0 ? 2 * g.w : 1));
    {
        const size_t lpO = border_lp_doubles(g, 2 * g.w, DK + 1), lpT = border_lp_doubles(g, g.w, 1);
        AL(p->LP, (lpO > lpT ? lpO : lpT) + 1);
    }
    AL(p->gamA, (size_t)(DK + 1) * (DB + 1) * L * ny);
    AL(p->gam, (size_t)g.NK * g.NB * L * L);
    AL(p->gamP, (size_t)((ny + 255) / 256) * g.NK * g.NB * L * L);
    AL(p->phi, g.NB * g.NB);
    AL(p->delta, g.NB);
    for (int i = 1; i < NSCI; i++) AL(p->deltax[i], g.NB);
    AL(p->G, (size_t)n * n);
    if (e == cudaSuccess) { e = cudaMalloc(&p->gmeta, (size_t)n * sizeof(int)); if (e == cudaSuccess) p->bytes += (size_t)n * sizeof(int); }
    AL(p->h, n);
    AL(p->Lf, (size_t)n * n);
    AL(p->dscale, n);
    AL(p->Linv, (size_t)((n + 63) / 64) * 64 * 64);
    AL(p->ywork, 2 * (size_t)(((n + 63) / 64) * 64)); // flag-in-data exchange words of the triangular solves (two per element)
    AL(p->zwork, 2 * (size_t)(((n + 63) / 64) * 64));
    AL(p->coef, n);
    for (int i = 1; i < 2 * NSCI; i++) { AL(p->hq[i], n); AL(p->cq[i], n); }
    AL(p->E, (size_t)g.NK * L * (g.Hx + 1));
    AL(p->wcorr, (size_t)(2LL * g.w * nx + 2LL * g.w * (ny - 2 * g.w)) + 1);
    AL(p->flag, 2);   // [0] pivot test failed (factorisation), [1] triangular-solve error
#undef AL
    p->specTo = p->specT;
    if (e == cudaSuccess) e = cudaMallocHost((void **)&p->flag_host, 2 * sizeof(int));
    if (e != cudaSuccess) {
        const bool oom = (e == cudaErrorMemoryAllocation);
        cudaGetLastError(); free_plan(p);
        return oom ? SFFT_ERR_ALLOC : SFFT_ERR_CUDA;
    }
    p->flag_host[0] = p->flag_host[1] = 0;
    for (int s = 0; s < SFFT_NUM_STAGES; s++) { cudaEventCreate(&p->ev0[s]); cudaEventCreate(&p->ev1[s]); }
    p->stream = 0; p->cur = 0;
    cudaStreamCreateWithFlags(&p->side, cudaStreamNonBlocking);
    cudaStreamCreateWithFlags(&p->sideB, cudaStreamNonBlocking);
    cudaStreamCreateWithFlags(&p->sideC, cudaStreamNonBlocking);
    cudaEventCreateWithFlags(&p->ev_joinB, cudaEventDisableTiming);
    cudaEventCreateWithFlags(&p->ev_joinC, cudaEventDisableTiming);
    cudaEventCreateWithFlags(&p->ev_fork, cudaEventDisableTiming);
    cudaEventCreateWithFlags(&p->ev_join, cudaEventDisableTiming);
    {   // highest priority: the factorisation is a chain of small dependent launches; its CTAs should take
        // the next free SM slots rather than queue behind the full-grid kernels of the science side
        int lo = 0, hi = 0;
        cudaDeviceGetStreamPriorityRange(&lo, &hi);
        cudaStreamCreateWithPriority(&p->fstream, cudaStreamNonBlocking, hi);
    }
    cudaEventCreateWithFlags(&p->ev_ffork, cudaEventDisableTiming);
    cudaStreamCreateWithFlags(&p->cstream, cudaStreamNonBlocking);
    cudaEventCreateWithFlags(&p->ev_copy, cudaEventDisableTiming);
    cudaEventCreateWithFlags(&p->ev_fjoin, cudaEventDisableTiming);
    {
        int lo = 0, hi = 0;
        cudaDeviceGetStreamPriorityRange(&lo, &hi);
        cudaStreamCreateWithPriority(&p->fstream2, cudaStreamNonBlocking, hi);
    }
    cudaEventCreateWithFlags(&p->ev_lookP, cudaEventDisableTiming);
    cudaEventCreateWithFlags(&p->ev_lookB, cudaEventDisableTiming);
    twiddle_kernel<<<(g.Nt + 255) / 256, 256>>>(p->tw, g.Nt);
    e = assemble_init(p);
    if (e == cudaSuccess) e = rows_init(p);
    if (e == cudaSuccess) e = cols_init();
    if (e == cudaSuccess) e = lags_init(p);   // tensor maps over the spectra, phase tables (after the twiddles)
    if (e != cudaSuccess) { cudaGetLastError(); free_plan(p); return SFFT_ERR_CUDA; }
    // Phi (pin P7): closed form, mask independent
    double phi[MAX_NP * MAX_NP];
    for (int s = 0; s < g.NB; s++)
        for (int s2 = 0; s2 < g.NB; s2++)
            phi[s * g.NB + s2] = power_sum(nx, g.pi[s] + g.pi[s2]) * power_sum(ny, g.pj[s] + g.pj[s2]);
    e = cudaMemcpy(p->phi, phi, sizeof(double) * g.NB * g.NB, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemset(p->flag, 0, 2 * sizeof(int));
    if (e == cudaSuccess) e = cudaMemset(p->ywork, 0, sizeof(double) * 2 * (size_t)(((n + 63) / 64) * 64)); // epoch 0 never matches a solve
    if (e == cudaSuccess) e = cudaMemset(p->zwork, 0, sizeof(double) * 2 * (size_t)(((n + 63) / 64) * 64));
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    if (e != cudaSuccess) { cudaGetLastError(); free_plan(p); return SFFT_ERR_CUDA; }
    p->launches = 1;
    *out = p;
    return SFFT_OK;
}

sfft_status sfft_plan_set_stream(sfft_plan *p, void *cuda_stream) {
    if (!p) return SFFT_ERR_INVALID_ARG;
    p->stream = (cudaStream_t)cuda_stream; p->cur = p->stream;
    return SFFT_OK;
}

sfft_status sfft_plan_destroy(sfft_plan *p) {
    if (!p) return SFFT_OK;
    join_factor(p);
    cudaStreamSynchronize(p->stream);
    free_plan(p);
    return SFFT_OK;
}

int sfft_num_unknowns(const sfft_plan *p) { return p ? p->g.n : 0; }
size_t sfft_workspace_bytes(const sfft_plan *p) { return p ? p->bytes : 0; }
long long sfft_launch_count(const sfft_plan *p) { return p ? p->launches : 0; }
const char *sfft_last_error(const sfft_plan *p) { return p ? p->err : "null plan"; }

} // extern "C"

// ------------------------------------------------------------------------------------------
// stage sequencing
// ------------------------------------------------------------------------------------------

// f4, constant photometric ratio: z_k = G^-1 e_k behind the factorisation on stream st (kept while the factor lives)
static cudaError_t ratio_Z(sfft_plan *p, cudaStream_t st) {
    const int m = p->g.NK - 1;
    if (m < 1) { p->have_ratioZ = true; return cudaSuccess; }
    if (!p->ratioEZ) { cudaError_t e = dalloc(p, &p->ratioEZ, (size_t)2 * m * p->g.n); if (e != cudaSuccess) return e; }
    if (m > 1 && !p->ratioW) { // first use: exchange words (epoch 0 never matches a solve), streams and events of the parallel solves
        const size_t cnt = (size_t)(m - 1) * 4 * (size_t)(((p->g.n + 63) / 64) * 64);
        cudaError_t e = dalloc(p, &p->ratioW, cnt);
        if (e == cudaSuccess) e = cudaMemsetAsync(p->ratioW, 0, cnt * sizeof(double), st); // ordered before the fork event of the solves
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->ev_rfork, cudaEventDisableTiming);
        for (int k = 0; k < m - 1 && e == cudaSuccess; k++) {
            int lo = 0, hi = 0;
            cudaDeviceGetStreamPriorityRange(&lo, &hi);
            e = cudaStreamCreateWithPriority(&p->rstream[k], cudaStreamNonBlocking, hi); // like the factor stream: latency chains go first
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->ev_rjoin[k], cudaEventDisableTiming);
        }
        if (e != cudaSuccess) return e;
    }
    cudaError_t e = launch_ratio_Z(p, p->ratioEZ, p->ratioEZ + (size_t)m * p->g.n, st, p->ratioW);
    if (e == cudaSuccess) p->have_ratioZ = true;
    return e;
}
static cudaError_t ratio_apply(sfft_plan *p, double *c, cudaStream_t st) {
    const int m = p->g.NK - 1;
    if (m < 1) return cudaSuccess;
    return launch_ratio_apply(p, p->ratioEZ + (size_t)m * p->g.n, c, st);
}

// a1 (template), Omega, Gamma, G.  Needs p->R, p->mask set.
static sfft_status template_side(sfft_plan *p) {
    const Geom &g = p->g;
    {
        StageTimer tm(p, SFFT_STAGE_A1_TEMPLATE);
        if (p->mask && p->specTo == p->specT) { // the subtraction needs spectra of the UNMASKED template (C7): allocated with the first mask
            const size_t nb = (size_t)g.NK * g.My * (g.Hx + 1) * p->spec_esz;
            CK(cudaMalloc(&p->specTo, nb), "alloc unmasked spectra");
            p->bytes += nb;
        }
        if (p->mask) {
            CK(launch_row_fwd(p, p->R, nullptr, p->inter, g.DK + 1, nullptr, 0), "row_fwd(R unmasked)");
            CK(launch_col_fwd(p, p->inter, p->specTo, g.NK, g.pi, g.pj), "col_fwd(R unmasked)");
        }
        CK(launch_row_fwd(p, p->R, p->mask, p->inter, g.DK + 1, p->muR, g.DK + g.DB + 1), "row_fwd(R)");
        CK(launch_col_fwd(p, p->inter, p->specT, g.NK, g.pi, g.pj), "col_fwd(R)");
    }
    {
        StageTimer tm(p, SFFT_STAGE_A2_OMEGA);
        fork_side(p);
        use_side(p, 2);
        CK(launch_gamma(p), "gamma");           // on a side stream, beside the Omega column pass
        back_to_main(p);
        CK(launch_lags(p, p->plO, 2 * g.w, p->lagO, false), "lags(Omega)"); // joins the side stream
    }
    {
        StageTimer tm(p, SFFT_STAGE_A3_GATHER);
        CK(launch_gather_G(p), "gather G");
    }
    return SFFT_OK;
}

// a1 (science), Theta, Delta, h.  Needs p->S (and p->R, p->mask of the template).
static sfft_status science_side(sfft_plan *p) {
    const Geom &g = p->g;
    {
        StageTimer tm(p, SFFT_STAGE_A1_SCIENCE);
        const int i0 = 0, j0 = 0;
        CK(launch_row_fwd(p, p->S, p->mask, p->inter, 1, p->muS, g.DB + 1), "row_fwd(S)");
        CK(launch_col_fwd(p, p->inter, p->specS, 1, &i0, &j0), "col_fwd(S)");
    }
    {
        StageTimer tm(p, SFFT_STAGE_A2_THETA);
        fork_side(p);
        use_side(p, 2);
        CK(launch_delta(p), "delta");
        back_to_main(p);
        CK(launch_lags(p, p->plT, g.w, p->lagT, true), "lags(Theta)");
        CK(launch_gather_h(p), "gather h");
    }
    return SFFT_OK;
}

// The same for nimg <= NSCI science images in ONE pass over the template spectra (batched path): a1 of each image, then
// one Theta lag pass with nimg NK pairs over NK + nimg spectra -- the NK template spectra are read once for the
// group ((NK + nimg)/nimg r per image instead of (NK + 1) r).  Results: hout[i].
static sfft_status science_sideN(sfft_plan *p, int nimg, const double *const *S, double *const *hout) {
    const Geom &g = p->g;
    p->muSx[0] = p->muS; p->deltax[0] = p->delta;
    const int i0 = 0, j0 = 0;
    for (int i = 0; i < nimg; i++) {
        p->Sx[i] = S[i];
        CK(launch_row_fwd(p, S[i], p->mask, p->inter, 1, p->muSx[i], g.DB + 1), "row_fwd(S)");
        CK(launch_col_fwd(p, p->inter, p->specSx[i], 1, &i0, &j0), "col_fwd(S)");
    }
    p->S = S[0];
    PairList pl; pl.np = nimg * g.NK;
    for (int q = 0; q < MAX_PAIRS; q++) pl.ord[q] = q;
    for (int i = 0; i < nimg; i++)
        for (int t = 0; t < g.NK; t++) { pl.a[i * g.NK + t] = t; pl.b[i * g.NK + t] = g.NK + i; }
    fork_side(p);
    use_side(p, 2);
    for (int i = 0; i < nimg; i++) CK(launch_delta(p, p->muSx[i], p->deltax[i]), "delta");
    back_to_main(p);
    CK(launch_lags(p, pl, g.w, p->lagT, true, nimg), "lags(Theta, several images)");
    for (int i = 0; i < nimg; i++)
        CK(launch_gather_h(p, p->lagT + (size_t)i * g.NK * g.L * g.L, p->deltax[i], hout[i]), "gather h");
    return SFFT_OK;
}

extern "C" {

sfft_status sfft_build_system(sfft_plan *p, const double *S, const double *R, const uint8_t *mask) {
    if (!p) return SFFT_ERR_INVALID_ARG;
    if (!S || !R) return fail(p, SFFT_ERR_INVALID_ARG, "build_system: NULL image");
    join_factor(p); // a factorisation still in flight reads G
    p->S = S; p->R = R; p->mask = mask;
    p->have_template = p->have_system = p->have_factor = p->have_solution = false;
    sfft_status st = template_side(p);
    if (st != SFFT_OK) return st;
    if (!p->ktiming && p->fstream && !p->knob.no_factor_overlap) {
        // G depends on the template only: factor it (a4) on its own stream while the science side (a1, Theta)
        // runs on the caller's stream; sfft_solve joins.
        fork_factor(p);
        {
            StageTimer tm(p, SFFT_STAGE_A4_FACTOR);
            CK(launch_factor(p), "factor");
            p->have_ratioZ = false;
            if (p->ratio_mode) CK(ratio_Z(p, p->cur), "constant-ratio solves");
        }
        back_to_main(p);
        p->have_factor = true;
    }
    if (p->science_waits_copy) { // sfft_difference_host: S is still on its way over PCIe (copy stream)
        CK(cudaStreamWaitEvent(p->stream, p->ev_copy, 0), "wait for the S upload");
        p->science_waits_copy = false;
    }
    st = science_side(p);
    if (st != SFFT_OK) return st;
    p->have_template = true; p->have_system = true;
    return SFFT_OK;
}

sfft_status sfft_solve(sfft_plan *p) {
    if (!p) return SFFT_ERR_INVALID_ARG;
    if (!p->have_system) return fail(p, SFFT_ERR_STATE, "solve before build_system");
    join_factor(p);
    if (!p->have_factor) {
        StageTimer tm(p, SFFT_STAGE_A4_FACTOR);
        CK(launch_factor(p), "factor");
        p->have_factor = true; p->have_ratioZ = false;
    }
    {
        StageTimer tm(p, SFFT_STAGE_A4_SOLVE);
        if (p->ratio_mode && !p->have_ratioZ) CK(ratio_Z(p, p->stream), "constant-ratio solves");
        CK(launch_trisolve(p, p->h, p->coef), "trisolve");
        if (p->ratio_mode) CK(ratio_apply(p, p->coef, p->stream), "constant-ratio correction");
    }
    p->have_solution = true;
    return SFFT_OK;
}

sfft_status sfft_set_constant_ratio(sfft_plan *p, int on) {
    if (!p) return SFFT_ERR_INVALID_ARG;
    p->ratio_mode = on != 0;
    return SFFT_OK;
}

sfft_status sfft_solve_constant_ratio(sfft_plan *p) {
    if (!p) return SFFT_ERR_INVALID_ARG;
    const bool saved = p->ratio_mode;
    p->ratio_mode = true;
    const sfft_status st = sfft_solve(p);
    p->ratio_mode = saved;
    return st;
}

sfft_status sfft_subtract(sfft_plan *p, double *D, double *coeffs) {
    if (!p) return SFFT_ERR_INVALID_ARG;
    if (!p->have_solution) return fail(p, SFFT_ERR_STATE, "subtract before solve");
    if (!D) return fail(p, SFFT_ERR_INVALID_ARG, "subtract: NULL D");
    {
        StageTimer tm(p, SFFT_STAGE_A5_SUBTRACT);
        CK(launch_subtract(p, p->S, p->R, p->coef, D), "subtract");
    }
    if (coeffs) CK(cudaMemcpyAsync(coeffs, p->coef, sizeof(double) * p->g.n, cudaMemcpyDeviceToDevice, p->stream), "copy coeffs");
    return SFFT_OK;
}

sfft_status sfft_subtract_with(sfft_plan *p, const double *S, const double *coeffs_in, double *D) {
    if (!p) return SFFT_ERR_INVALID_ARG;
    if (!p->have_template) return fail(p, SFFT_ERR_STATE, "subtract_with before build_system/set_template");
    if (!coeffs_in || !D) return fail(p, SFFT_ERR_INVALID_ARG, "subtract_with: NULL pointer");
    const double *Suse = S ? S : p->S;
    if (!Suse) return fail(p, SFFT_ERR_INVALID_ARG, "subtract_with: no science image");
    StageTimer tm(p, SFFT_STAGE_A5_SUBTRACT);
    CK(launch_subtract(p, Suse, p->R, coeffs_in, D), "subtract_with");
    return SFFT_OK;
}

// f2: out = img (*) stamp, circular at the native grid, through the a1/a5 kernels:
// row + column transform of the unweighted image into the science-spectrum buffer, K^ synthesised from the L x L
// taps, inverse transforms, wrap correction of the border pixels.  Geom is passed to kernels by value, so one
// spectrum / no background is a temporary NK = 1, NB = 0, DK = 0 view of the plan's geometry.
sfft_status sfft_convolve_stamp(sfft_plan *p, const double *img, const double *stamp, double *out) {
    if (!p) return SFFT_ERR_INVALID_ARG;
    if (!img || !stamp || !out) return fail(p, SFFT_ERR_INVALID_ARG, "convolve_stamp: NULL pointer");
    if (img == out) return fail(p, SFFT_ERR_INVALID_ARG, "convolve_stamp: in-place operation is not supported");
    back_to_main(p);
    const Geom saved = p->g;
    p->g.NK = 1; p->g.NB = 0; p->g.DK = 0; p->g.DB = 0;
    const int i0 = 0, j0 = 0;
    cudaError_t e = launch_row_fwd(p, img, nullptr, p->inter, 1, nullptr, 0);
    if (e == cudaSuccess) e = launch_col_fwd(p, p->inter, p->specS, 1, &i0, &j0);
    if (e == cudaSuccess) e = launch_subtract(p, nullptr, img, stamp, out, p->specS, 1);
    p->g = saved;
    CK(e, "convolve_stamp");
    return SFFT_OK;
}

static bool affine_ok(const double *M) {
    if (!M) return false;
    for (int i = 0; i < 6; i++) if (!(M[i] - M[i] == 0.0)) return false; // NaN or infinite
    return true;
}

sfft_status sfft_resample_affine(sfft_plan *p, const double *img, const double *M, int method, double fill, double *out) {
    if (!p) return SFFT_ERR_INVALID_ARG;
    if (!img || !out) return fail(p, SFFT_ERR_INVALID_ARG, "resample_affine: NULL pointer");
    if (img == out) return fail(p, SFFT_ERR_INVALID_ARG, "resample_affine: in-place operation is not supported");
    if (!affine_ok(M)) return fail(p, SFFT_ERR_INVALID_ARG, "resample_affine: the matrix must be 6 finite numbers");
    if (method != 0 && method != 1 && method != 3) return fail(p, SFFT_ERR_INVALID_ARG, "resample_affine: method must be 0 (nearest), 1 (bilinear) or 3 (Lanczos-3)");
    back_to_main(p);
    CK(launch_resample(p, img, M, method, fill, out), "resample_affine");
    return SFFT_OK;
}

sfft_status sfft_resample_affine_mask(sfft_plan *p, const uint8_t *mask, const double *M, int fill, uint8_t *out) {
    if (!p) return SFFT_ERR_INVALID_ARG;
    if (!mask || !out) return fail(p, SFFT_ERR_INVALID_ARG, "resample_affine_mask: NULL pointer");
    if (mask == out) return fail(p, SFFT_ERR_INVALID_ARG, "resample_affine_mask: in-place operation is not supported");
    if (!affine_ok(M)) return fail(p, SFFT_ERR_INVALID_ARG, "resample_affine_mask: the matrix must be 6 finite numbers");
    if (fill < 0 || fill > 255) return fail(p, SFFT_ERR_INVALID_ARG, "resample_affine_mask: fill must be 0..255");
    back_to_main(p);
    CK(launch_resample_mask(p, mask, M, fill, out), "resample_affine_mask");
    return SFFT_OK;
}

sfft_status sfft_local_kernel(sfft_plan *p, const double *coeffs, double x, double y, double *K_out) {
    if (!p) return SFFT_ERR_INVALID_ARG;
    if (!K_out) return fail(p, SFFT_ERR_INVALID_ARG, "local_kernel: NULL output");
    if (!coeffs) {
        if (!p->have_solution) return fail(p, SFFT_ERR_STATE, "local_kernel: no coefficients given and nothing solved yet");
        coeffs = p->coef;
    }
    if (!(x == x) || !(y == y)) return fail(p, SFFT_ERR_INVALID_ARG, "local_kernel: position is NaN");
    back_to_main(p);
    const double xt = (2.0 * x + 1.0 - p->g.nx) / (double)p->g.nx, yt = (2.0 * y + 1.0 - p->g.ny) / (double)p->g.ny; // reading C3
    CK(launch_local_kernel(p, coeffs, xt, yt, K_out), "local_kernel");
    return SFFT_OK;
}

sfft_status sfft_decorrelation_stamp(sfft_plan *p, const double *K, int Lk, const double *psf_S, const double *psf_R,
                                     int Lp, double var_S, double var_R, int N, double *stamp_out) {
    if (!p) return SFFT_ERR_INVALID_ARG;
    if (!K || !psf_S || !psf_R || !stamp_out) return fail(p, SFFT_ERR_INVALID_ARG, "decorrelation_stamp: NULL pointer");
    if (Lk < 1 || Lp < 1 || !(Lk & 1) || !(Lp & 1)) return fail(p, SFFT_ERR_INVALID_ARG, "decorrelation_stamp: stamp sizes must be odd and >= 1");
    if (N > 1024 || N < Lk + Lp - 1 || N < Lp || N < p->g.L) return fail(p, SFFT_ERR_INVALID_ARG, "decorrelation_stamp: need max(Lk + Lp - 1, L) <= N <= 1024");
    if (!(var_S >= 0.0) || !(var_R >= 0.0) || !(var_S + var_R > 0.0) || var_S + var_R > 1.7e308)
        return fail(p, SFFT_ERR_INVALID_ARG, "decorrelation_stamp: variances must be finite, >= 0 and not both 0");
    const size_t have = (size_t)(p->g.DK + 1) * p->g.My * p->g.Hx * sizeof(cplx), need = ((size_t)N * N + 1) * sizeof(double);
    if (need > have) return fail(p, SFFT_ERR_INVALID_ARG, "decorrelation_stamp: N x N grid does not fit the plan's intermediate buffer");
    join_factor(p);
    back_to_main(p);
    double *F = reinterpret_cast<double *>(p->inter);
    int *bad = reinterpret_cast<int *>(F + (size_t)N * N);
    CK(launch_decorr(p, K, Lk, psf_S, psf_R, Lp, var_S, var_R, N, F, bad, stamp_out), "decorrelation_stamp");
    int bad_host = 0;
    CK(cudaMemcpyAsync(&bad_host, bad, sizeof(int), cudaMemcpyDeviceToHost, p->stream), "decorrelation_stamp: read flag");
    CK(cudaStreamSynchronize(p->stream), "decorrelation_stamp: sync");
    if (bad_host) return fail(p, SFFT_ERR_INVALID_ARG, "decorrelation_stamp: the noise power spectrum has a zero (or overflowed): the kernel is undefined");
    return SFFT_OK;
}

sfft_status sfft_set_template(sfft_plan *p, const double *R, const uint8_t *mask) {
    if (!p) return SFFT_ERR_INVALID_ARG;
    if (!R) return fail(p, SFFT_ERR_INVALID_ARG, "set_template: NULL image");
    join_factor(p);
    p->R = R; p->mask = mask; p->S = nullptr;
    p->have_template = p->have_system = p->have_factor = p->have_solution = false;
    sfft_status st = template_side(p);
    if (st != SFFT_OK) return st;
    {
        StageTimer tm(p, SFFT_STAGE_A4_FACTOR);
        CK(launch_factor(p), "factor");
        p->have_ratioZ = false;
        if (p->ratio_mode) CK(ratio_Z(p, p->cur), "constant-ratio solves");
    }
    p->have_template = true; p->have_factor = true;
    return SFFT_OK;
}

sfft_status sfft_subtract_batch(sfft_plan *p, const double *const *S, int B, double *const *D, double *coeffs) {
    if (!p) return SFFT_ERR_INVALID_ARG;
    if (!p->have_template || !p->have_factor) return fail(p, SFFT_ERR_STATE, "subtract_batch before set_template");
    if (!S || !D || B < 1) return fail(p, SFFT_ERR_INVALID_ARG, "subtract_batch: bad arguments");
    for (int b = 0; b < B; b++) if (!S[b] || !D[b]) return fail(p, SFFT_ERR_INVALID_ARG, "subtract_batch: NULL image");
    join_factor(p); // the factor may come from sfft_build_system's overlap path and still be in flight on the factor stream
    if (B > 1 && !p->timing && !p->ktiming && p->fstream && !p->knob.no_batch_pipe) {
        // Groups of up to NSCI images per science-side pass (science_sideN), and a software pipeline over the groups: the
        // triangular solves of group k (latency-bound launches that leave the machine empty) run on the factor stream
        // beside the science-side kernels of group k+1.  Order on the main stream: sci(0), [sci(1), a5(group 0)],
        // [sci(2), a5(group 1)], ...  h and the coefficients are buffered per (group parity, image); the solves of group
        // k+2 start after sci(k+2), which is behind a5(group k) on the main stream, so no buffer is overwritten while in use.
        p->hq[0] = p->h; p->cq[0] = p->coef;
        const int gsz = p->knob.batch_group;
        const int ngrp = (B + gsz - 1) / gsz;
        auto sci = [&](int k) -> sfft_status {
            const int b0 = gsz * k, nimg = B - b0 < gsz ? B - b0 : gsz;
            return science_sideN(p, nimg, S + b0, p->hq + NSCI * (k & 1));
        };
        if (p->ratio_mode && !p->have_ratioZ) CK(ratio_Z(p, p->stream), "constant-ratio solves");
        sfft_status rc = sci(0);
        if (rc == SFFT_OK) CK(cudaEventRecord(p->ev_ffork, p->stream), "event");
        for (int k = 0; k < ngrp && rc == SFFT_OK; k++) {
            const int b0 = gsz * k, nimg = B - b0 < gsz ? B - b0 : gsz, par = NSCI * (k & 1);
            cudaStreamWaitEvent(p->fstream, p->ev_ffork, 0);
            cudaError_t e = cudaSuccess;
            for (int i = 0; i < nimg && e == cudaSuccess; i++) {
                e = launch_trisolve(p, p->hq[par + i], p->cq[par + i], p->fstream);
                if (e == cudaSuccess && p->ratio_mode) e = ratio_apply(p, p->cq[par + i], p->fstream);
            }
            if (e == cudaSuccess) e = cudaEventRecord(p->ev_fjoin, p->fstream);
            CK(e, "trisolve (batch)");
            if (k + 1 < ngrp) {
                rc = sci(k + 1);
                if (rc != SFFT_OK) break;
                cudaEventRecord(p->ev_ffork, p->stream);
            }
            cudaStreamWaitEvent(p->stream, p->ev_fjoin, 0);
            for (int i = 0; i < nimg && e == cudaSuccess; i++) {
                e = launch_subtract(p, S[b0 + i], p->R, p->cq[par + i], D[b0 + i]);
                if (e == cudaSuccess && coeffs)
                    e = cudaMemcpyAsync(coeffs + (size_t)(b0 + i) * p->g.n, p->cq[par + i], sizeof(double) * p->g.n, cudaMemcpyDeviceToDevice, p->stream);
            }
            CK(e, "subtract (batch)");
        }
        if (rc != SFFT_OK) return rc;
        // leave the plan as the sequential path does: S, h, coef = those of the last image
        const int last = NSCI * ((ngrp - 1) & 1) + (B - 1 - gsz * (ngrp - 1));
        if (last != 0) {
            cudaMemcpyAsync(p->h, p->hq[last], sizeof(double) * p->g.n, cudaMemcpyDeviceToDevice, p->stream);
            cudaMemcpyAsync(p->coef, p->cq[last], sizeof(double) * p->g.n, cudaMemcpyDeviceToDevice, p->stream);
        }
        p->S = S[B - 1];
        p->have_system = p->have_solution = true;
        return SFFT_OK;
    }
    for (int b = 0; b < B; b++) {
        p->S = S[b];
        sfft_status st = science_side(p);
        if (st != SFFT_OK) return st;
        p->have_system = true;
        {
            StageTimer tm(p, SFFT_STAGE_A4_SOLVE);
            if (p->ratio_mode && !p->have_ratioZ) CK(ratio_Z(p, p->stream), "constant-ratio solves");
            CK(launch_trisolve(p, p->h, p->coef), "trisolve");
            if (p->ratio_mode) CK(ratio_apply(p, p->coef, p->stream), "constant-ratio correction");
        }
        p->have_solution = true;
        {
            StageTimer tm(p, SFFT_STAGE_A5_SUBTRACT);
            CK(launch_subtract(p, p->S, p->R, p->coef, D[b]), "subtract");
        }
        if (coeffs)
            CK(cudaMemcpyAsync(coeffs + (size_t)b * p->g.n, p->coef, sizeof(double) * p->g.n, cudaMemcpyDeviceToDevice, p->stream), "copy coeffs");
    }
    return SFFT_OK;
}

sfft_status sfft_sync_status(sfft_plan *p) {
    if (!p) return SFFT_ERR_INVALID_ARG;
    join_factor(p);
    CK(cudaStreamSynchronize(p->stream), "sync");
    if (p->side) { CK(cudaStreamSynchronize(p->side), "sync side"); CK(cudaStreamSynchronize(p->sideB), "sync side"); CK(cudaStreamSynchronize(p->sideC), "sync side"); }
    if (p->have_factor) {
        CK(cudaMemcpy(p->flag_host, p->flag, 2 * sizeof(int), cudaMemcpyDeviceToHost), "read flag");
        if (p->flag_host[1]) {   // the coefficients of that solve are NaN (sfft_solve.cu: ll_load); clear so the plan stays usable
            CK(cudaMemset(p->flag + 1, 0, sizeof(int)), "clear solve flag");
            return fail(p, SFFT_ERR_CUDA, "triangular solve: a solution block never arrived");
        }
        if (p->flag_host[0]) return fail(p, SFFT_ERR_NOT_SPD, "pivot <= 1e-12: matrix not positive definite");
    }
    return SFFT_OK;
}

sfft_status sfft_difference_host(sfft_plan *p, const double *S_host, const double *R_host, const uint8_t *mask_host,
                                 double *D_host, double *coeffs_host) {
    if (!p) return SFFT_ERR_INVALID_ARG;
    if (!S_host || !R_host || !D_host) return fail(p, SFFT_ERR_INVALID_ARG, "difference_host: NULL buffer");
    const size_t npix = (size_t)p->g.nx * p->g.ny;
    if (!p->stS) {
        CK(dalloc(p, &p->stS, npix), "alloc staging"); CK(dalloc(p, &p->stR, npix), "alloc staging");
        CK(dalloc(p, &p->stD, npix), "alloc staging");
    }
    if (mask_host && !p->stM) CK(dalloc(p, &p->stM, npix), "alloc staging");
    // R (and the mask) first on the caller's stream; S follows on the copy stream and overlaps the template-side
    // a1/a2 (the previous call ended with a full synchronisation, so the staging buffers are free)
    if (mask_host) CK(cudaMemcpyAsync(p->stM, mask_host, npix, cudaMemcpyHostToDevice, p->stream), "H2D mask");
    CK(cudaMemcpyAsync(p->stR, R_host, npix * sizeof(double), cudaMemcpyHostToDevice, p->stream), "H2D R");
    CK(cudaEventRecord(p->ev_copy, p->stream), "order the S upload after the R upload");
    CK(cudaStreamWaitEvent(p->cstream, p->ev_copy, 0), "order the S upload");
    CK(cudaMemcpyAsync(p->stS, S_host, npix * sizeof(double), cudaMemcpyHostToDevice, p->cstream), "H2D S");
    CK(cudaEventRecord(p->ev_copy, p->cstream), "H2D S done");
    p->science_waits_copy = true;
    sfft_status st = sfft_build_system(p, p->stS, p->stR, mask_host ? p->stM : nullptr);
    if (st == SFFT_OK) st = sfft_solve(p);
    if (st == SFFT_OK) st = sfft_subtract(p, p->stD, nullptr);
    if (st != SFFT_OK) return st;
    CK(cudaMemcpyAsync(D_host, p->stD, npix * sizeof(double), cudaMemcpyDeviceToHost, p->stream), "D2H D");
    if (coeffs_host) CK(cudaMemcpyAsync(coeffs_host, p->coef, sizeof(double) * p->g.n, cudaMemcpyDeviceToHost, p->stream), "D2H coeffs");
    return sfft_sync_status(p);
}


// e2e for configs[3]: one template, B science images, all in HOST memory.  The template goes up once; the images run
// through a three-deep pipeline  H2D(S_{i+1}) | compute(i) | D2H(D_{i-1})  on two plan-owned copy streams beside the
// caller's stream, one plain cudaMemcpyAsync per buffer (PCIe is full duplex: the upload of the next image and the
// download of the previous result overlap each other and the ~0.6 ms of device work).
sfft_status sfft_difference_host_batch(sfft_plan *p, const double *R_host, const uint8_t *mask_host, const double *const *S_host,
                                       int B, double *const *D_host, double *coeffs_host) {
    if (!p) return SFFT_ERR_INVALID_ARG;
    if (!R_host || !S_host || !D_host || B < 1) return fail(p, SFFT_ERR_INVALID_ARG, "difference_host_batch: bad arguments");
    for (int b = 0; b < B; b++) if (!S_host[b] || !D_host[b]) return fail(p, SFFT_ERR_INVALID_ARG, "difference_host_batch: NULL image");
    const size_t npix = (size_t)p->g.nx * p->g.ny, n = p->g.n;
    constexpr int NSLOT = 3;
    if (!p->hbS[0]) { // first use: staging buffers, the download stream, events
        if (!p->stR) CK(dalloc(p, &p->stR, npix), "alloc staging");
        for (int k = 0; k < NSLOT; k++) {
            CK(dalloc(p, &p->hbS[k], npix), "alloc staging"); CK(dalloc(p, &p->hbD[k], npix), "alloc staging");
            CK(dalloc(p, &p->hbC[k], n), "alloc staging");
            CK(cudaEventCreateWithFlags(&p->ev_hin[k], cudaEventDisableTiming), "event");
            CK(cudaEventCreateWithFlags(&p->ev_hcomp[k], cudaEventDisableTiming), "event");
            CK(cudaEventCreateWithFlags(&p->ev_hout[k], cudaEventDisableTiming), "event");
        }
        CK(cudaStreamCreateWithFlags(&p->ostream, cudaStreamNonBlocking), "stream");
    }
    if (mask_host && !p->stM) CK(dalloc(p, &p->stM, npix), "alloc staging");
    // the first science image starts up beside the template
    CK(cudaEventRecord(p->ev_copy, p->stream), "event");       // everything enqueued before this call is done with the buffers
    CK(cudaStreamWaitEvent(p->cstream, p->ev_copy, 0), "wait");
    CK(cudaStreamWaitEvent(p->ostream, p->ev_copy, 0), "wait");
    if (mask_host) CK(cudaMemcpyAsync(p->stM, mask_host, npix, cudaMemcpyHostToDevice, p->stream), "H2D mask");
    CK(cudaMemcpyAsync(p->stR, R_host, npix * sizeof(double), cudaMemcpyHostToDevice, p->stream), "H2D R");
    sfft_status st = sfft_set_template(p, p->stR, mask_host ? p->stM : nullptr);
    if (st != SFFT_OK) return st;
    for (int b = 0; b < B; b++) {
        const int k = b % NSLOT;
        if (b >= NSLOT) CK(cudaStreamWaitEvent(p->cstream, p->ev_hcomp[k], 0), "wait"); // image b-3 no longer reads hbS[k]
        CK(cudaMemcpyAsync(p->hbS[k], S_host[b], npix * sizeof(double), cudaMemcpyHostToDevice, p->cstream), "H2D S");
        CK(cudaEventRecord(p->ev_hin[k], p->cstream), "event");
        CK(cudaStreamWaitEvent(p->stream, p->ev_hin[k], 0), "wait");
        if (b >= NSLOT) CK(cudaStreamWaitEvent(p->stream, p->ev_hout[k], 0), "wait");   // D of image b-3 has left hbD[k], hbC[k]
        const double *Sd = p->hbS[k]; double *Dd = p->hbD[k];
        st = sfft_subtract_batch(p, &Sd, 1, &Dd, p->hbC[k]);
        if (st != SFFT_OK) return st;
        CK(cudaEventRecord(p->ev_hcomp[k], p->stream), "event");
        CK(cudaStreamWaitEvent(p->ostream, p->ev_hcomp[k], 0), "wait");
        CK(cudaMemcpyAsync(D_host[b], p->hbD[k], npix * sizeof(double), cudaMemcpyDeviceToHost, p->ostream), "D2H D");
        if (coeffs_host) CK(cudaMemcpyAsync(coeffs_host + (size_t)b * n, p->hbC[k], n * sizeof(double), cudaMemcpyDeviceToHost, p->ostream), "D2H coeffs");
        CK(cudaEventRecord(p->ev_hout[k], p->ostream), "event");
    }
    CK(cudaStreamSynchronize(p->ostream), "sync downloads");
    return sfft_sync_status(p);
}

} // extern "C"

// ------------------------------------------------------------------------------------------
// introspection
// ------------------------------------------------------------------------------------------
extern "C" {

sfft_status sfft_get_system(const sfft_plan *pc, double *G, double *h) {
    sfft_plan *p = const_cast<sfft_plan *>(pc);
    if (!p) return SFFT_ERR_INVALID_ARG;
    if (!p->have_template) return fail(p, SFFT_ERR_STATE, "get_system: nothing built yet");
    const size_t n = p->g.n;
    if (G) CK(cudaMemcpyAsync(G, p->G, n * n * sizeof(double), cudaMemcpyDeviceToDevice, p->stream), "copy G");
    if (h) {
        if (!p->have_system) return fail(p, SFFT_ERR_STATE, "get_system: no right-hand side yet");
        CK(cudaMemcpyAsync(h, p->h, n * sizeof(double), cudaMemcpyDeviceToDevice, p->stream), "copy h");
    }
    return SFFT_OK;
}

sfft_status sfft_enable_timings(sfft_plan *p, int on) {
    if (!p) return SFFT_ERR_INVALID_ARG;
    p->timing = on == 1;
    p->ktiming = on == 2;
    p->nkrec = 0;
    for (int s = 0; s < SFFT_NUM_STAGES; s++) p->ev_used[s] = false;
    return SFFT_OK;
}

int sfft_kernel_timing_count(const sfft_plan *p) { return p ? p->nkrec : 0; }

sfft_status sfft_kernel_timing_get(sfft_plan *p, int i, const char **name, float *ms) {
    if (!p || !name || !ms || i < 0 || i >= p->nkrec) return SFFT_ERR_INVALID_ARG;
    CK(cudaEventSynchronize(p->krec[i].e1), "sync");
    *name = p->krec[i].name; *ms = 0.0f;
    CK(cudaEventElapsedTime(ms, p->krec[i].e0, p->krec[i].e1), "elapsed");
    return SFFT_OK;
}

sfft_status sfft_get_timings(sfft_plan *p, float *ms, int n_stages) {
    if (!p || !ms || n_stages < 0) return SFFT_ERR_INVALID_ARG;
    CK(cudaStreamSynchronize(p->stream), "sync");
    for (int s = 0; s < n_stages; s++) {
        ms[s] = 0.0f;
        if (s < SFFT_NUM_STAGES && p->ev_used[s]) {
            float t = 0.0f;
            if (cudaEventElapsedTime(&t, p->ev0[s], p->ev1[s]) == cudaSuccess) ms[s] = t; else cudaGetLastError();
        }
    }
    return SFFT_OK;
}

sfft_status sfft_debug_read(sfft_plan *p, int which, int idx, void *host_dst, size_t nbytes) {
    if (!p || !host_dst) return SFFT_ERR_INVALID_ARG;
    const Geom &g = p->g;
    const size_t plane = (size_t)g.My * (g.Hx + 1) * sizeof(cplx), dplane = (size_t)g.My * (g.Hx + 1) * p->spec_esz;
    const int W2 = 4 * g.w + 1, LL = g.L * g.L;
    const void *src = nullptr; size_t sz = 0;
    double dims[2] = {(double)g.Mx, (double)g.My};
    switch (which) {
    case 0: if (idx < 0 || idx >= g.NK) return SFFT_ERR_INVALID_ARG; src = (const char *)p->specT + (size_t)idx * dplane; sz = plane; break;
    case 1: src = p->specS; sz = plane; break;
    case 2: if (idx < 0 || idx >= p->npairsO) return SFFT_ERR_INVALID_ARG; src = p->lagO + (size_t)idx * W2 * W2; sz = sizeof(double) * W2 * W2; break;
    case 3: if (idx < 0 || idx >= g.NK) return SFFT_ERR_INVALID_ARG; src = p->lagT + (size_t)idx * LL; sz = sizeof(double) * LL; break;
    case 4: src = p->gam; sz = sizeof(double) * g.NK * g.NB * LL; break;
    case 5: src = p->phi; sz = sizeof(double) * g.NB * g.NB; break;
    case 6: src = p->delta; sz = sizeof(double) * g.NB; break;
    case 7: if (nbytes != sizeof(dims)) return SFFT_ERR_INVALID_ARG; memcpy(host_dst, dims, sizeof(dims)); return SFFT_OK;
    case 8: src = p->inter; sz = (size_t)g.My * g.Hx * sizeof(cplx); break; // plane 0 of the intermediates, raw [Hx][My]
    default: return SFFT_ERR_INVALID_ARG;
    }
    if (nbytes != sz) return fail(p, SFFT_ERR_INVALID_ARG, "debug_read: size mismatch");
    CK(cudaStreamSynchronize(p->stream), "sync");
    if (which <= 1) { // spectra are column-major on the device (plane_idx), complex128 or complex64: hand them out as [My][Hx+1] complex128
        void *tmp = malloc(dplane);
        if (!tmp) return fail(p, SFFT_ERR_ALLOC, "debug_read: host allocation failed");
        cudaError_t e = cudaMemcpy(tmp, src, dplane, cudaMemcpyDeviceToHost);
        if (e == cudaSuccess)
            for (int ky = 0; ky < g.My; ky++)
                for (int kx = 0; kx <= g.Hx; kx++) {
                    const size_t i = plane_idx(ky, kx, g.My);
                    ((cplx *)host_dst)[(size_t)ky * (g.Hx + 1) + kx] = p->spec32 ? ld_c(((const float2 *)tmp)[i]) : ((const cplx *)tmp)[i];
                }
        free(tmp);
        CK(e, "debug copy");
        return SFFT_OK;
    }
    CK(cudaMemcpy(host_dst, src, sz, cudaMemcpyDeviceToHost), "debug copy");
    return SFFT_OK;
}

sfft_status sfft_probe_fp64(int kind, int iters, double *tflops) {
    if (!tflops || iters < 1 || kind < 0 || kind > 1) return SFFT_ERR_INVALID_ARG;
    return run_probe_fp64(kind, iters, tflops) == cudaSuccess ? SFFT_OK : SFFT_ERR_CUDA;
}

} // extern "C"
