// sfft_internal.h -- plan layout and kernel launchers shared by the .cu files of libsfft.
// Not part of the C ABI (include/sfft.h is).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include "../../include/sfft.h"
#include "sfft_fft.cuh"

namespace sfft {

constexpr int MAX_DEG = 3;                                   // DK, DB <= 3
constexpr int MAX_NP = (MAX_DEG + 1) * (MAX_DEG + 2) / 2;    // 10 polynomial terms
constexpr int MAX_L = 21;
constexpr int NSCI = 4;    // science images per Theta pass of the batched path
constexpr int MAX_PAIRS = MAX_NP * (MAX_NP + 1) / 2;         // 55 unordered template pairs
constexpr double PIVOT_MIN = 1e-12;                          // reading C9

// Geometry every kernel needs, passed by value.
struct Geom {
    int nx, ny;        // frame
    int Mx, My;        // zero-padded power-of-two FFT sizes
    int Hx;            // Mx/2: complex columns of a (packed) half spectrum
    int log2Hx, log2My;
    int L, w;          // kernel size, half width
    int DK, DB, NK, NB, n;
    int Nt;            // twiddle table length (max(Mx, My)); tw[k] = exp(-2 pi i k/Nt)
    int pi[MAX_NP], pj[MAX_NP]; // t -> (i,j): total degree ascending, then j ascending
};

constexpr int MAX_KREC = 512;  // per-launch timing records kept between two sfft_enable_timings calls
struct KRec { const char *name; cudaEvent_t e0, e1; };

struct PairList {           // spectra pairs (A = spec[a[p]], B = spec[b[p]]) of one lag pass
    int np;
    int a[MAX_PAIRS], b[MAX_PAIRS];
    int ord[MAX_PAIRS];     // thread slot -> pair: self-pairs (a == b) first, so that they fill whole warps of the lag pass
};

// launch shape of stage 1 of a lag pass (sfft_lags.cu), fixed at plan creation
struct LagCfg { int WB, KXC, npg, nkb, ngr, nsplit, halves, rows_per_split, nst; bool wide; size_t smem; }; // wide: one CTA of <= 384 threads per SM
struct LagMaps;             // TMA tensor maps of a lag pass (sfft_lags.cu)
} // namespace sfft
struct CUtensorMap_st;      // <cuda.h>: CUtensorMap
namespace sfft {

// Experiment knobs (environment variables SFFT_*), read ONCE at sfft_plan_create: nothing on the hot path calls getenv
struct Knobs {
    bool no_side;           // SFFT_NO_SIDE: keep the small kernels on the caller's stream
    bool no_factor_overlap; // SFFT_NO_FACTOR_OVERLAP: factor inside sfft_solve instead of beside the science side
    bool no_batch_pipe;     // SFFT_NO_BATCH_PIPE: sequential batched path
    bool no_lookahead;      // SFFT_NO_LOOKAHEAD: trailing updates of the Cholesky on the chain's own stream
    int batch_group;        // SFFT_BATCH_GROUP: science images per Theta pass (1..NSCI)
    int factor_sms;         // SFFT_FACTOR_SMS: SMs the persistent column kernels leave to a factorisation running beside them
};

} // namespace sfft

struct sfft_plan {
    sfft::Geom g;
    cudaStream_t stream;     // the caller's stream: every call is ordered on it
    cudaStream_t side;       // plan-owned: small independent kernels run beside the big ones (fork/join by events)
    cudaStream_t sideB, sideC; // two more, so that the independent small chains (packed column | wrap corrections |
    cudaEvent_t ev_joinB, ev_joinC; // Gamma/Delta) also run beside EACH OTHER: each is latency-bound on a small grid
    cudaStream_t cur;        // stream the launchers enqueue on right now (stream, or side inside a fork)
    cudaEvent_t ev_fork, ev_join;
    cudaStream_t fstream;    // plan-owned: the factorisation of a single pair runs here, beside the science-side a1/a2
    cudaEvent_t ev_ffork, ev_fjoin;
    cudaStream_t fstream2;   // look-ahead of the blocked Cholesky: the rest of a trailing update runs here
    cudaEvent_t ev_lookP, ev_lookB;
    cudaStream_t cstream;    // plan-owned copy stream: sfft_difference_host uploads S here while the template side computes
    cudaEvent_t ev_copy; bool science_waits_copy;
    sfft::Knobs knob;        // experiment knobs, read once at plan creation
    int sms;                 // multiprocessors of the plan's device
    bool factor_pending;     // factor kernels are enqueued on fstream and not yet joined into `stream`
    bool lf_ready;           // Lf, dscale hold the equilibrated G already (written by the gather of G): launch_factor skips that step
    // device workspaces
    sfft::cplx *tw;          // [Nt]
    sfft::cplx *rtw;         // [3][Hx/16] the row passes' per-thread twiddles, compact (sfft_rows.cu: rowtw_kernel)
    // planes are column-major (sfft_fft.cuh: plane_idx): intermediates [Hx][My] (column 0 packed), spectra [Hx+1][My]
    sfft::cplx *inter;       // [(DK+1)][Hx][My] row-transformed intermediates (a1) / a5 intermediate
    // spectrum elements are complex128, or complex64 in the reduced-memory plan mode (spec32; arithmetic stays FP64)
    bool spec32; size_t spec_esz; // element size in bytes: 16 or 8
    void *specT;             // [NK][Hx+1][My] spectra of the fit (masked) template images
    void *specTo;            // [NK][Hx+1][My] spectra of the unmasked template images (allocated with the first mask)
    void *specS;             // [Hx+1][My]
    // batched path: up to NSCI science images share one Theta pass; groups of images are pipelined two deep
    void *specSx[sfft::NSCI]; // [Hx+1][My] each; [0] aliases specS
    double *muSx[sfft::NSCI], *deltax[sfft::NSCI]; // row moments / Delta per image; [0] alias muS, delta
    double *hq[2 * sfft::NSCI], *cq[2 * sfft::NSCI]; // right-hand sides / solutions: group parity x image; [0] alias h, coef
    const double *Sx[sfft::NSCI];   // the science images of the current group
    double *muR;             // [(DK+DB+1)][ny] row moments sum_x xt^m (m.R)
    double *muS;             // [(DB+1)][ny]
    sfft::cplx *Q;           // [split][np][2W+1][Hx+1] column-reduced products (stage 1 of a2)
    sfft::cplx *phO, *phT;   // phase tables of the lag passes (sfft_lags.cu: lag_phase_kernel)
    sfft::LagCfg cfgO, cfgT[sfft::NSCI]; // launch shapes: Omega; Theta with 1..NSCI science images
    sfft::LagMaps *mapsO, *mapsT;        // their tensor maps (host copies, passed to the kernels by value)
    CUtensorMap_st *mapI;                // tensor map of the a5 intermediate (sfft_rows.cu)
    double *lagO;            // [npairs][(4w+1)^2]
    double *lagT;            // [NK][L*L]
    double *bpart;           // [np][(2W+1)^2] native-grid wrap corrections X_N - X_M
    double *SB;              // [2 images][4 sides][W][max(nx,ny)] border strips of m.R, m.S (sfft_border.cu)
    double *LP;              // [chunk][4][W][W][2W+1][DK+1][DK+1|1] line-pair linear correlations
    double *gamA;            // [(DK+1)][(DB+1)][L][ny] row sums for Gamma
    double *gam;             // [NK][NB][L*L]
    double *gamP;            // [ceil(ny/256)][NK][NB][L*L] chunk partials of Gamma (sfft_assemble.cu)
    double *phi;             // [NB][NB]
    double *delta;           // [NB]
    double *G;               // [n][n]
    int *gmeta;              // [n] index meta data of the unknowns for the gather of G (sfft_assemble.cu)
    double *h;               // [n]
    double *h2, *coef2;      // [n] each: second right-hand side / solution (the batched path pipelines two images)
    double *Lf;              // [n][n] Cholesky factor of the equilibrated matrix (lower, row-major)
    double *dscale;          // [n]   1/sqrt(G_ii)
    double *Linv;            // [nblk][64][64] inverses of the factor's diagonal blocks
    double *ywork, *zwork;   // [n] forward / backward substitution vectors
    int solve_epoch;         // epoch tag of the flag-in-data exchange words of the triangular solves (ywork, zwork), one per solve
    double *coef;            // [n]   solved coefficients
    double *ratioEZ;         // [2][NK-1][n] indicator right-hand sides and their solves (sfft_solve_constant_ratio; allocated on first use)
    sfft::cplx *E;           // [NK][L][Hx+1] kernel row tables for a5
    double *wcorr;           // [border pixels] native-grid wrap corrections of a5 (sfft_subtract.cu)
    int *flag;               // device: 1 = pivot test failed
    int *flag_host;          // pinned mirror
    // host staging for sfft_difference_host
    double *stS, *stR, *stD; uint8_t *stM;
    // sfft_difference_host_batch: three-deep upload | compute | download pipeline (allocated on first use)
    double *hbS[3], *hbD[3], *hbC[3]; cudaStream_t ostream; cudaEvent_t ev_hin[3], ev_hcomp[3], ev_hout[3];
    size_t bytes;
    // state
    const double *S, *R; const uint8_t *mask;
    bool have_template, have_system, have_factor, have_solution;
    bool ratio_mode;         // sfft_set_constant_ratio: every solve is followed by the constant-ratio correction
    bool have_ratioZ;        // ratioEZ holds the z_k of the current factor
    double *ratioW;          // [NK-2][2][2*ceil64(n)] exchange words of the auxiliary solves 2..NK-1, which run beside the first
    cudaStream_t rstream[sfft::MAX_NP - 2]; cudaEvent_t ev_rfork, ev_rjoin[sfft::MAX_NP - 2];
    int npairsO;
    sfft::PairList plO, plT;
    // timing
    bool timing; cudaEvent_t ev0[SFFT_NUM_STAGES], ev1[SFFT_NUM_STAGES]; bool ev_used[SFFT_NUM_STAGES];
    // per-launch timing (sfft_enable_timings(plan, 2)): one event pair per kernel launch, in launch order
    bool ktiming; int nkrec; sfft::KRec krec[sfft::MAX_KREC];
    long long launches;
    char err[256];
};

namespace sfft {

// ---- a1, a5 transforms (sfft_rows.cu, sfft_cols.cu) -------------------------------------------
cudaError_t rows_init(sfft_plan *p);   // kernel attributes of the current device, tensor map of the a5 intermediate (plan creation)
void rows_free(sfft_plan *p);
cudaError_t cols_init();
// rows: img (ny x nx real, optional mask) -> inter[i] ([Hx][My]), i = 0..NI-1, weights xt^i;
// also row moments mu[m][y] = sum_x xt^m (m.img), m = 0..NMOM-1.
cudaError_t launch_row_fwd(sfft_plan *p, const double *img, const uint8_t *mask, cplx *inter, int NI,
                           double *mu, int NMOM);
// columns: FFT_y(yt^jj[k] * inter[ii[k]]) -> spec[k] ([Hx+1][My]), k = 0..ns-1
cudaError_t launch_col_fwd(sfft_plan *p, const cplx *inter, void *spec, int ns, const int *ii, const int *jj);
// inter = IFFT_y(sum_t spec_t K^_t(coef))
cudaError_t launch_col_inv(sfft_plan *p, const void *spec, const double *coef, cplx *inter);
// mode 0: D = S - M - B; mode 1: D = +M
cudaError_t launch_row_inv(sfft_plan *p, const cplx *inter, const double *S, const double *coef, double *D, int mode);

int border_chunks();
int border_linpair_chunks();
size_t border_lp_doubles(const Geom &g, int W, int EB);
size_t border_strip_doubles(const Geom &g, int W);
cudaError_t launch_border(sfft_plan *p, const PairList &pl, int W, bool science, double *bpart);
// ---- a2, a3 (sfft_lags.cu, sfft_assemble.cu) ---------------------------------------------------------
void lagcol_config(const Geom &g, int np, int ns, int W, LagCfg *c, size_t esz); // esz: bytes per spectrum element
cudaError_t lags_init(sfft_plan *p);   // launch shapes, tensor maps, phase tables (plan creation, after the spectra exist)
void lags_free(sfft_plan *p);
size_t lag_q_elems(const sfft_plan *p);
// lag tables of pair list pl over the template spectra (index < NK) and, for science passes, specSx[i] (index NK + i)
cudaError_t launch_lags(sfft_plan *p, const PairList &pl, int W, double *lag /*[np][(2W+1)^2]*/, bool science, int nsci = 1);
// nsci > 1: pl lists the NK pairs of each image in turn (images p->Sx[i])
cudaError_t launch_gamma(sfft_plan *p);   // muR, R, mask -> gam
cudaError_t launch_delta(sfft_plan *p, const double *muS = nullptr, double *delta = nullptr);   // muS -> delta
cudaError_t assemble_init(sfft_plan *p);
cudaError_t launch_gather_G(sfft_plan *p);
cudaError_t launch_gather_h(sfft_plan *p, const double *lagT = nullptr, const double *delta = nullptr, double *h = nullptr);

// ---- a4 (sfft_solve.cu) ------------------------------------------------------------------
cudaError_t launch_factor(sfft_plan *p);                      // G -> dscale, Lf, flag
cudaError_t launch_trisolve(sfft_plan *p, const double *h, double *c, cudaStream_t st = nullptr, double *work = nullptr); // c = D (L^-T (L^-1 (D h))); st: default the plan's stream; work: own exchange words [2][2*ceil64(n)] (zeroed once) for a solve that runs beside another one, default the plan's

// ---- a5 (sfft_subtract.cu) ---------------------------------------------------------------
// spec: the NK spectra to convolve (default: the plan's unmasked template spectra); mode 0: D = S - M - B,
// mode 1 (f2, sfft_convolve_stamp): D = +M, S unused
cudaError_t launch_subtract(sfft_plan *p, const double *S, const double *R, const double *coef, double *D,
                            const void *spec = nullptr, int mode = 0);

// ---- f1 (sfft_decorr.cu) -----------------------------------------------------------------
cudaError_t launch_local_kernel(sfft_plan *p, const double *coef, double xt, double yt, double *K);
// F: N*N doubles of scratch, bad: one int (raised when the noise power is not positive somewhere)
cudaError_t launch_decorr(sfft_plan *p, const double *K, int Lk, const double *PS, const double *PR, int Lp,
                          double varS, double varR, int N, double *F, int *bad, double *stamp);

// ---- f4 constant photometric ratio (sfft_ratio.cu) ---------------------------------------
// E, Z: [NK-1][n] each: indicator right-hand sides and z_k = G^-1 e_k (factor only); apply: c free solution in,
// constrained solution out
cudaError_t launch_ratio_Z(sfft_plan *p, double *E, double *Z, cudaStream_t st, double *W);
cudaError_t launch_ratio_apply(sfft_plan *p, const double *Z, double *c, cudaStream_t st);

// ---- f3 (sfft_align.cu) ------------------------------------------------------------------
// M: 6 host doubles (output pixel -> source position); method 0 nearest, 1 bilinear, 3 Lanczos-3
cudaError_t launch_resample(sfft_plan *p, const double *img, const double *M, int method, double fill, double *out);
cudaError_t launch_resample_mask(sfft_plan *p, const uint8_t *mask, const double *M, int fill, uint8_t *out);

// ---- probes (sfft_probe.cu) -------------------------------------------------------------------
cudaError_t run_probe_fp64(int kind, int iters, double *tflops);

// RAII around ONE kernel launch: counts it and, in per-launch timing mode, brackets it with events.
struct KLaunch {
    sfft_plan *p; KRec *r;
    KLaunch(sfft_plan *p_, const char *name) : p(p_), r(nullptr) {
        p->launches++;
        if (p->ktiming && p->nkrec < MAX_KREC) {
            r = &p->krec[p->nkrec];
            if (!r->e0) { cudaEventCreate(&r->e0); cudaEventCreate(&r->e1); }
            r->name = name; p->nkrec++;
            cudaEventRecord(r->e0, p->cur);
        }
    }
    ~KLaunch() { if (r) cudaEventRecord(r->e1, p->cur); }
};

// side stream: fork = side waits for everything enqueued on the main stream so far; join = main waits for side.
// In per-launch timing mode everything stays on the main stream so that kernel times do not overlap.
inline void fork_side(sfft_plan *p) {
    if (p->ktiming || !p->side || p->knob.no_side) return;
    cudaEventRecord(p->ev_fork, p->stream);
    cudaStreamWaitEvent(p->side, p->ev_fork, 0); cudaStreamWaitEvent(p->sideB, p->ev_fork, 0); cudaStreamWaitEvent(p->sideC, p->ev_fork, 0);
    p->cur = p->side;
}
inline void use_side(sfft_plan *p, int k) { // after fork_side: enqueue on side stream k (0, 1, 2)
    if (p->ktiming || !p->side || p->knob.no_side) return;
    p->cur = k == 0 ? p->side : k == 1 ? p->sideB : p->sideC;
}
inline void back_to_main(sfft_plan *p) { p->cur = p->stream; }
inline void join_side(sfft_plan *p) {
    p->cur = p->stream;
    if (p->ktiming || !p->side || p->knob.no_side) return;
    cudaEventRecord(p->ev_join, p->side); cudaStreamWaitEvent(p->stream, p->ev_join, 0);
    cudaEventRecord(p->ev_joinB, p->sideB); cudaStreamWaitEvent(p->stream, p->ev_joinB, 0);
    cudaEventRecord(p->ev_joinC, p->sideC); cudaStreamWaitEvent(p->stream, p->ev_joinC, 0);
}

// the factorisation stream: same fork/join protocol as the side stream
inline void fork_factor(sfft_plan *p) {
    cudaEventRecord(p->ev_ffork, p->stream); cudaStreamWaitEvent(p->fstream, p->ev_ffork, 0);
    p->cur = p->fstream; p->factor_pending = true;
}
inline void join_factor(sfft_plan *p) {
    p->cur = p->stream;
    if (!p->factor_pending) return;
    cudaEventRecord(p->ev_fjoin, p->fstream); cudaStreamWaitEvent(p->stream, p->ev_fjoin, 0);
    p->factor_pending = false;
}

inline int ilog2(int v) { int l = 0; while ((1 << l) < v) l++; return l; }

} // namespace sfft
