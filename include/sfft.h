/*
 * sfft.h -- C ABI of libsfft: the SFFT (Saccadic Fast Fourier Transform) subtraction
 * hot path on one NVIDIA B200 (sm_100a), FP64.
 *
 * What the library computes (BASELINE.json north_star; the paper only names the method:
 * PAPER.md:29 "Saccadic Fast Fourier Transform (SFFT) method for difference imaging",
 * PAPER.md:43 "flexible delta basis function", "[GPU] Apply SFFT subtraction"):
 *
 *     D = S - (R (*) K(x,y)) - B(x,y)
 *
 * K is an L x L delta-basis kernel whose coefficients vary as a 2-D polynomial of total
 * degree DK over the frame, B a background polynomial of total degree DB.  The
 * n = L*L*NK + NB coefficients (NK=(DK+1)(DK+2)/2, NB=(DB+1)(DB+2)/2) are the linear
 * least-squares solution of  min || vec(m.S) - A c ||_2 ; column (t,u,v) of A is the
 * image (x,y) -> T_t((x-u) mod nx, (y-v) mod ny),  T_t = xt^i yt^j (m.R),  column s is
 * P_s = xt^p yt^q  (not masked);  xt = (2x+1-nx)/nx, yt = (2y+1-ny)/ny;  boundary
 * conditions are circular at the native nx x ny (readings C2-C7).
 *
 * Steps:
 *   a1  polynomial-weighted template images and their 2-D FFTs      (sfft_build_system)
 *   a2  cross-correlations at kernel-offset pairs from the spectra   (sfft_build_system)
 *   a3  gather into G = A^T A (n x n) and h = A^T b                  (sfft_build_system)
 *   a4  FP64 Cholesky solve of the Jacobi-equilibrated system        (sfft_solve)
 *   a5  FFT convolution with the solved kernel + fused subtraction   (sfft_subtract)
 *   a6  batched: one template, many science images                  (sfft_set_template,
 *                                                                     sfft_subtract_batch)
 *
 * Conventions
 *   - images: row-major FP64, img[y*nx + x], 0 <= x < nx, 0 <= y < ny, DEVICE pointers
 *     unless a parameter says "host"; inputs are never modified.
 *   - mask: DEVICE ny*nx uint8 (non-zero = use pixel in the fit) or NULL = all ones.
 *     The fit uses m.S and m.R; the subtraction uses the unmasked S and R.
 *   - coefficient layout (output of the method), w = (L-1)/2:
 *       coeffs[t*L*L + (v+w)*L + (u+w)] = a_{t,u,v},  t <-> (i,j) in the order
 *       (0,0),(1,0),(0,1),(2,0),(1,1),(0,2),(3,0),...  (total degree ascending, then j);
 *       coeffs[NK*L*L + s] = b_s in the same (p,q) order.
 *     The kernel applied at SOURCE pixel (x',y') is K(u,v) = sum_t a_{t,u,v} xt(x')^i yt(y')^j.
 *   - every call enqueues its kernels on the plan's CUDA stream and returns without
 *     synchronising the device, except where stated.  No exceptions cross the boundary;
 *     every function returns an sfft_status (or a plain value for the getters).
 *   - the plan owns all workspaces (twiddles, spectra, lag tables, G, the factor).
 *   - there is NO CPU fallback: without a CUDA device sfft_plan_create fails with
 *     SFFT_ERR_CUDA.
 */
#ifndef SFFT_H
#define SFFT_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sfft_plan sfft_plan; /* opaque */

typedef enum {
    SFFT_OK = 0,
    SFFT_ERR_INVALID_ARG = -1, /* bad size / NULL pointer / unsupported L or frame size       */
    SFFT_ERR_ALLOC = -2,       /* host or device allocation failed                             */
    SFFT_ERR_CUDA = -3,        /* a CUDA runtime call or kernel launch failed (no device etc.) */
    SFFT_ERR_STATE = -4,       /* call order: solve before build, subtract before solve, ...   */
    SFFT_ERR_NOT_SPD = -5      /* a pivot of the equilibrated matrix was <= 1e-12 (reading C9) */
} sfft_status;

/* Stage indices of sfft_get_timings (milliseconds of the most recent call of each stage). */
enum {
    SFFT_STAGE_A1_TEMPLATE = 0, /* weighted template images + forward FFTs           */
    SFFT_STAGE_A1_SCIENCE = 1,  /* forward FFT of m.S                                */
    SFFT_STAGE_A2_OMEGA = 2,    /* template-template lag tables (+Gamma)             */
    SFFT_STAGE_A2_THETA = 3,    /* template-science lag tables (+Delta)              */
    SFFT_STAGE_A3_GATHER = 4,   /* fill of G and h                                   */
    SFFT_STAGE_A4_FACTOR = 5,   /* equilibration + Cholesky factorisation            */
    SFFT_STAGE_A4_SOLVE = 6,    /* two triangular solves                             */
    SFFT_STAGE_A5_SUBTRACT = 7, /* kernel spectrum synthesis, inverse FFTs, D        */
    SFFT_NUM_STAGES = 8
};

#define SFFT_MAX_SIDE 4096

/* Create a plan for nx x ny frames, L x L kernel (L odd, 1 <= L <= 21), polynomial degrees
 * DK, DB (0 <= DK, DB <= 3).  Requires 2L-1 <= nx, ny <= SFFT_MAX_SIDE (4096: the Roman
 * detector frame is 4088 x 4088).  Frames are zero-padded internally to powers
 * of two (at least 1024 x 512) and the sums that wrap differently on the padded grid are
 * corrected exactly, so any nx, ny in range is supported, including 256, 1024 and 4088.
 * Allocates every workspace (nothing is allocated later except the second set of template
 * spectra on the first call with a mask and the host-path staging buffers); uses the
 * current CUDA device and the legacy default stream until sfft_plan_set_stream.
 * Errors: INVALID_ARG, ALLOC, CUDA (no usable device). */
sfft_status sfft_plan_create(sfft_plan **out, int nx, int ny, int L, int DK, int DB);

/* The same with option flags.  SFFT_PLAN_FP32_SPECTRA: the reduced-memory mode (PAPER.md:105, 113 name GPU memory as
 * the barrier) -- the spectra (the plan's largest buffers: NK + 4 planes) are STORED as complex64,
 * all arithmetic and every other buffer stay FP64.  Halves the spectrum memory and the bytes the lag passes and the
 * subtraction read; the loosened tolerances this costs are stated as numbers in DESIGN.md (reduced-memory mode) and
 * asserted by tests/test_gpu_fp32_spectra.py.  Unknown flag bits: INVALID_ARG. */
#define SFFT_PLAN_FP32_SPECTRA 1u
sfft_status sfft_plan_create_ex(sfft_plan **out, int nx, int ny, int L, int DK, int DB, unsigned flags);

/* cuda_stream is a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream). */
sfft_status sfft_plan_set_stream(sfft_plan *plan, void *cuda_stream);

/* Synchronises the plan's stream, frees everything.  NULL is accepted. */
sfft_status sfft_plan_destroy(sfft_plan *plan);

/* n = L*L*NK + NB (BASELINE.json north_star: unknown count).  0 for a NULL plan. */
int sfft_num_unknowns(const sfft_plan *plan);

/* Bytes of device memory the plan holds.  0 for a NULL plan. */
size_t sfft_workspace_bytes(const sfft_plan *plan);

/* ---- single pair ------------------------------------------------------------------ */

/* a1-a3 for one (S, R, mask): afterwards the plan holds G and h.  The plan keeps the
 * POINTERS S and R (not copies) for sfft_subtract: both must stay alive and unchanged
 * until sfft_subtract has been enqueued and has run.  Errors: INVALID_ARG (NULL S/R), CUDA. */
sfft_status sfft_build_system(sfft_plan *plan, const double *S, const double *R,
                              const uint8_t *mask);

/* a4: Jacobi equilibration, blocked Cholesky, two triangular solves.  Asynchronous: a
 * failed pivot test is recorded on the device and reported by sfft_sync_status (or by the
 * next sfft_subtract with a host coefficient read).  Errors: STATE, CUDA. */
sfft_status sfft_solve(sfft_plan *plan);

/* f4 variant ("constant-photometric-ratio constraint (drops the sum-flux freedom of higher-order
 * terms)"; reading R1 of DESIGN.md section 15): sfft_solve, then the solution is replaced by the least-squares solution
 * subject to  sum_{u,v} a_{t,u,v} = 0  for every polynomial term t = 1..NK-1, so that the flux scaling sum_{u,v} K(u,v;x,y)
 * is the same everywhere on the frame (term t = 0 and the background stay free).  Uses the factor of sfft_solve: NK-1
 * more pairs of triangular solves and an (NK-1) x (NK-1) Schur system.  DK = 0: identical to sfft_solve.  Allocates
 * 2 (NK-1) n doubles of plan workspace on first use.  sfft_subtract then uses the constrained coefficients.
 * Errors: those of sfft_solve; ALLOC / CUDA. */
sfft_status sfft_solve_constant_ratio(sfft_plan *plan);

/* The same constraint as a plan mode (on != 0): from now on EVERY solve of the plan -- sfft_solve, the per-image solves of
 * sfft_subtract_batch, sfft_difference_host -- is followed by the constant-ratio correction.  The NK-1 auxiliary solves
 * depend on the factor only: in this mode they are enqueued right behind the factorisation (on the plan's factor stream,
 * beside the science-side kernels; once per template in the batched path) and each solve then costs one small
 * correction kernel more.  Default: off.  Coefficients already solved are not changed.  Errors: INVALID_ARG (NULL plan). */
sfft_status sfft_set_constant_ratio(sfft_plan *plan, int on);

/* a5: D (device, ny*nx) = S - sum_t T_t (*) K_t - B using the solved coefficients;
 * coeffs (device, n doubles) receives them, or NULL.  Errors: STATE, INVALID_ARG, CUDA. */
sfft_status sfft_subtract(sfft_plan *plan, double *D, double *coeffs);

/* Debug/verification variant of a5: subtract with coefficients the
 * CALLER supplies (device, n doubles) instead of the solved ones.  Needs a prior
 * sfft_build_system or sfft_set_template (+ S given here when S != NULL).  */
sfft_status sfft_subtract_with(sfft_plan *plan, const double *S, const double *coeffs_in,
                               double *D);

/* ---- batched: one template, many science images (BASELINE.json configs[3]) ---------- */

/* Template-side work, once: a1 (template), Omega, Gamma, Phi, the matrix part of a3 and
 * the Cholesky factor of a4.  Keeps the pointer R (see sfft_build_system). */
sfft_status sfft_set_template(sfft_plan *plan, const double *R, const uint8_t *mask);

/* For b = 0..B-1: a1 (science), Theta, Delta, h, two triangular solves, a5.  The images go
 * through the Theta pass in groups of up to four (the template spectra are read once per group)
 * and the groups are pipelined against the solves; every image's result equals the single-pair
 * path's up to FP64 rounding.  The first batched call allocates up to three more science spectra
 * (ny_pad * nx_pad/2 complex each).
 * S, D: HOST arrays of B device pointers (ny*nx doubles each), all distinct from each other;
 * coeffs: device B*n doubles or NULL.  mask is the one given to sfft_set_template.
 * Errors: STATE, INVALID_ARG, CUDA. */
sfft_status sfft_subtract_batch(sfft_plan *plan, const double *const *S, int B,
                                double *const *D, double *coeffs);

/* ---- f2: cross-convolution with a PSF stamp (pipeline step 5: "Cross-convolve the
 * template PSF with the science image, and the science PSF with the template") ---------- */

/* out(x, y) = sum_{|u|,|v| <= w} stamp[(v + w) * L + (u + w)] * img((x - u) mod nx, (y - v) mod ny):
 * the discrete convolution of img (device, ny*nx doubles, row-major) with an L x L stamp (device, L*L
 * doubles, same tap layout as the kernel coefficients; L, w = (L-1)/2 are the plan's), circular at the
 * native nx x ny like the subtraction (reading C6).  out: device, ny*nx doubles, must not alias img.
 * Runs the a1 transforms of img, the a5 K^ synthesis / inverse transforms and the border wrap
 * correction; uses the plan's science-spectrum and intermediate buffers as scratch.  Both are dead between the
 * plan's calls (the intermediates live inside sfft_build_system / sfft_subtract, the science spectrum is consumed by
 * sfft_build_system and rebuilt per image by sfft_subtract_batch), and everything is ordered on the plan's stream, so
 * the call is allowed ANYWHERE in the call sequence, also between sfft_build_system and sfft_subtract
 * (tests/test_gpu_parity.py::test_scratch_users_between_build_and_subtract).  The plan's DK, DB are irrelevant.
 * Asynchronous on the plan's stream.
 * Errors: INVALID_ARG (NULL or aliased pointers), CUDA. */
sfft_status sfft_convolve_stamp(sfft_plan *plan, const double *img, const double *stamp, double *out);

/* ---- f3: alignment / resampling onto the science grid (pipeline step 4: "Align the reference image,
 * reference PSF, and reference detection mask to the science image").  PAPER.md names neither the
 * geometric model nor the interpolant; DESIGN.md section 14 lists the readings A1-A4 implemented here. ---------- */

/* out(x, y) = interpolant of img at xs = (M[0] x + M[1] y) + M[2], ys = (M[3] x + M[4] y) + M[5]  (the affine map from
 * an OUTPUT pixel to SOURCE pixel coordinates, pixel centres at integers, FP64, evaluated in this order without fused
 * multiply-add).  img, out: device, ny*nx doubles, row-major, the plan's frame size, must not alias.  M: HOST, 6 doubles
 * (read before the call returns).  method: 0 = nearest (pixel floor(xs + 0.5), floor(ys + 0.5)); 1 = bilinear;
 * 3 = Lanczos-3, k(t) = sinc(t) sinc(t/3), |t| < 3, the 6 weights of each axis divided by their sum.  An output pixel
 * whose footprint (taps floor(xs)-a+1 .. floor(xs)+a on each axis, a = 1 / 3; the one pixel for nearest) is not entirely
 * inside the frame is set to `fill` (any double, NaN allowed).  Touches no plan workspace (callable at any point of the
 * call sequence); asynchronous on the plan's stream.  The plan's L, DK, DB are irrelevant.
 * Errors: INVALID_ARG (NULL or aliased pointers, non-finite M, unknown method), CUDA. */
sfft_status sfft_resample_affine(sfft_plan *plan, const double *img, const double *M, int method, double fill,
                                 double *out);

/* The same geometry for a detection mask: nearest neighbour on uint8 (device, ny*nx), pixels from outside = fill
 * (0..255).  Errors: INVALID_ARG, CUDA. */
sfft_status sfft_resample_affine_mask(sfft_plan *plan, const uint8_t *mask, const double *M, int fill, uint8_t *out);

/* ---- f1: the decorrelation kernel (pipeline step 7: "Fit and apply the decorrelation kernel to
 * the difference image.  Also apply the decorrelation kernel to the science PSF and cross-convolved science image")
 * PAPER.md gives no formula; DESIGN.md section 13 lists the readings D1-D5 these two calls implement.  The kernel is
 * APPLIED with sfft_convolve_stamp (to D, to the cross-convolved science image; to the science PSF on a small plan). -- */

/* K_out[(v + w) * L + (u + w)] = sum_t a_{t,u,v} xt(x)^i yt(y)^j: the local matching kernel at pixel (x, y) of the
 * frame (reading D2; xt, yt the centred coordinates of reading C3; x, y may be fractional or outside the frame: the
 * polynomial is simply evaluated there).  coeffs: device, n doubles in the coefficient layout above, or NULL = the
 * plan's current solution (STATE error if there is none).  K_out: device, L*L doubles.  Asynchronous on the plan's
 * stream.  Errors: INVALID_ARG (NULL output, NaN position), STATE, CUDA. */
sfft_status sfft_local_kernel(sfft_plan *plan, const double *coeffs, double x, double y, double *K_out);

/* stamp_out = the central L x L taps (L the plan's) of the decorrelation kernel W,
 *     W^(k) = sqrt(F(0) / F(k)),  F(k) = var_S |P_R^(k)|^2 + var_R |P_S^(k)|^2 |K^(k)|^2,
 * transforms taken on an N x N periodic grid (readings D1, D3, D4): F is the noise power spectrum of
 * D = S (*) P_R - (R (*) P_S) (*) K for white pixel noise of variance var_S in S and var_R in R; W is real and even,
 * W^(0) = 1 (flux scale kept); the crop is not renormalised.
 * K: device, Lk*Lk doubles (e.g. from sfft_local_kernel); psf_S, psf_R: device, Lp*Lp doubles each; all stamps in
 * the tap layout stamp[(v + w) * P + (u + w)], P odd.  stamp_out: device, L*L doubles.
 * N: any integer with max(Lk + Lp - 1, L) <= N <= 1024 (no power-of-two restriction: the transforms are pruned direct
 * sums over the stamp taps); (N*N + 1) doubles of the plan's intermediate buffer serve as scratch (dead between the
 * plan's calls: allowed anywhere in the call sequence, like sfft_convolve_stamp).
 * SYNCHRONISES the plan's stream (a per-frame set-up call) and returns INVALID_ARG if F is zero, negative or not finite
 * at any grid frequency (the kernel is undefined there; stamp_out is then unspecified).
 * Errors: INVALID_ARG (NULL pointers, even or non-positive stamp sizes, N out of range or larger than the scratch,
 * negative / non-finite / both-zero variances, zero of F), CUDA. */
sfft_status sfft_decorrelation_stamp(sfft_plan *plan, const double *K, int Lk, const double *psf_S,
                                     const double *psf_R, int Lp, double var_S, double var_R, int N,
                                     double *stamp_out);

/* ---- host-buffer convenience (the end-to-end call bench.py times as `e2e`) ---------- */

/* Whole single-pair path from HOST buffers: copies S, R (and mask, may be NULL) to plan-owned
 * device staging, runs a1-a5, copies D (ny*nx) and coeffs (n, may be NULL) back and
 * SYNCHRONISES.  Returns NOT_SPD if the pivot test failed. */
sfft_status sfft_difference_host(sfft_plan *plan, const double *S_host, const double *R_host,
                                 const uint8_t *mask_host, double *D_host, double *coeffs_host);

/* The batched path (BASELINE.json configs[3]; every template against many science images; PAPER.md:101:
 * "holds all data in-memory to minimize time spent on file I/O") from HOST buffers: R_host (and mask_host, may be NULL)
 * go up once and sfft_set_template runs; then the B science images S_host[b] (HOST array of B host pointers, ny*nx
 * doubles each) stream through a three-deep pipeline -- upload of image b+1 | a1, Theta, solve, a5 of image b |
 * download of D of image b-1 -- on two plan-owned copy streams beside the plan's stream, one cudaMemcpyAsync per
 * buffer.  D_host[b]: B host pointers (ny*nx doubles each); coeffs_host: B*n doubles or NULL.  Pinned host memory is
 * needed for the copies to overlap.  Allocates seven frame-sized staging buffers on first use; SYNCHRONISES.
 * Errors: INVALID_ARG, ALLOC, CUDA, NOT_SPD. */
sfft_status sfft_difference_host_batch(sfft_plan *plan, const double *R_host, const uint8_t *mask_host,
                                       const double *const *S_host, int B, double *const *D_host, double *coeffs_host);

/* ---- introspection for tests and bench ------------------------------------------------ */

/* Synchronises the stream and returns SFFT_ERR_NOT_SPD if the most recent factorisation
 * failed its pivot test, SFFT_ERR_CUDA on a sticky CUDA error, else SFFT_OK. */
sfft_status sfft_sync_status(sfft_plan *plan);

/* Copies G (device, n*n, symmetric so row-major == column-major) and/or h (device, n);
 * either may be NULL.  Errors: STATE (nothing built yet). */
sfft_status sfft_get_system(const sfft_plan *plan, double *G, double *h);

/* Timing mode: 0 = off (default), 1 = per stage, 2 = per kernel launch.  Resets what was recorded.
 * sfft_get_timings: ms[0..n_stages) <- per-stage milliseconds (CUDA events on the plan's
 * stream) of the most recent call of each stage; synchronises.  */
sfft_status sfft_enable_timings(sfft_plan *plan, int on);
sfft_status sfft_get_timings(sfft_plan *plan, float *ms, int n_stages);

/* Mode 2: every kernel launch since sfft_enable_timings(plan, 2) is bracketed by a CUDA event
 * pair on the plan's stream (at most 512 are kept).  sfft_kernel_timing_count returns how many
 * were recorded; sfft_kernel_timing_get gives launch i's kernel name (static string, library
 * owned) and its milliseconds (synchronises on that launch).  Errors: INVALID_ARG, CUDA. */
int sfft_kernel_timing_count(const sfft_plan *plan);
sfft_status sfft_kernel_timing_get(sfft_plan *plan, int i, const char **name, float *ms);

/* Number of kernel launches this plan has enqueued since creation (bench: gpu_launches). */
long long sfft_launch_count(const sfft_plan *plan);

/* Plan-owned, NUL-terminated description of the most recent error ("" if none). */
const char *sfft_last_error(const sfft_plan *plan);

/* Library version string, e.g. "sfft-b200 0.1 (sm_100a)". */
const char *sfft_version(void);

/* Test hook: copies an internal device array to a HOST buffer (synchronises).
 *   which = 0: template spectrum t=idx  (My x (Hx+1) complex128, row-major [ky][kx], kx = 0..Hx = Mx/2)
 *           1: science spectrum
 *           2: Omega lag table of pair idx ((4w+1)^2 doubles, [dv+2w][du+2w])
 *           3: Theta lag table of t=idx (L*L doubles)
 *           4: Gamma (NK*NB*L*L doubles), 5: Phi (NB*NB), 6: Delta (NB)
 *           7: padded sizes {Mx, My} as two doubles
 * Returns INVALID_ARG if nbytes is not the array's size. */
sfft_status sfft_debug_read(sfft_plan *plan, int which, int idx, void *host_dst, size_t nbytes);

/* Allocation-free variant of step a4 (north_star (c), reading C9): solves G c = h by the
 * same kernels as sfft_solve (Jacobi equilibration, blocked Cholesky, the two triangular solves) WITHOUT a plan and
 * without allocating anything: no cudaMalloc / cudaFree, no stream or event creation, no allocating library call.
 * For callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid it).
 *   G  DEVICE, n x n doubles, row-major, symmetric positive definite; only the lower triangle (c <= r) is read
 *   h  DEVICE, n doubles          c  DEVICE, n doubles, written          (caller-owned; G and h are not modified)
 *   n  1 <= n <= SFFT_SOLVE_STATIC_MAX_N; larger n (or n < 1, or a NULL pointer) returns SFFT_ERR_INVALID_ARG and
 *      sfft_solve_static_last_error() names the limit
 *   cuda_stream  the cudaStream_t the work is ordered on (NULL = the default stream)
 * Scratch (the factor, the inverted diagonal blocks, the scaling, the exchange words of the triangular solves, the
 * flags: 8.6 MiB) lives in ONE file-scope `static __device__` array: every GPU that loads the library holds it until
 * the process exits.  Every call on a device shares it and it keeps the previous call's contents (the call clears
 * what must start at zero), so calls that overlap on the GPU -- two streams, two host threads -- RACE: serialise them.
 * The call BLOCKS until the solve has finished (it reads the pivot flag back) and returns SFFT_ERR_NOT_SPD if a pivot
 * of the equilibrated matrix was <= 1e-12 (c is then meaningless), SFFT_ERR_CUDA on a CUDA error or a lost exchange
 * block (c is then NaN-poisoned). */
#define SFFT_SOLVE_STATIC_MAX_N 1024
sfft_status sfft_solve_static(const double *G, const double *h, double *c, int n, void *cuda_stream);
/* Thread-local, NUL-terminated description of the calling thread's most recent sfft_solve_static error ("" if none). */
const char *sfft_solve_static_last_error(void);

/* FP64 rate probes used by bench.py to state the ALU roofline it divides by
 * (DESIGN.md "peaks"): runs a register-resident DFMA (kind=0) or DMMA m8n8k4 (kind=1)
 * loop on every SM for `iters` iterations and returns the achieved TFLOP/s in *tflops. */
sfft_status sfft_probe_fp64(int kind, int iters, double *tflops);

#ifdef __cplusplus
}
#endif
#endif /* SFFT_H */
