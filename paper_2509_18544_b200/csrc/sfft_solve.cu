// sfft_solve.cu -- step a4 (BASELINE.json north_star (c), reading C9):
// FP64 solve of G c = h.  G~ = D^-1/2 G D^-1/2 (D = diag G) is factored G~ = L L^T by a
// right-looking blocked Cholesky (block 64): diagonal block in one CTA, panel by triangular
// solve, trailing update C -= X X^T on the FP64 tensor pipe (mma.sync m8n8k4 f64 -- the one
// dense contraction of the path).  A pivot L_kk^2 <= 1e-12 raises the device flag
// (SFFT_ERR_NOT_SPD).  c = D^-1/2 L^-T L^-1 D^-1/2 h by two blocked triangular solves.
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <mutex>
#include "sfft_internal.h"

namespace sfft {

constexpr int CB = 64;      // Cholesky block
constexpr int CLD = CB + 4; // shared-memory leading dimension (conflict-free f64 fragment loads)

__global__ void equil_diag_kernel(const double *__restrict__ G, double *__restrict__ dscale, int n, int *flag) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double gii = G[(size_t)i * n + i];
    if (!(gii > 0.0)) { *flag = 1; dscale[i] = 1.0; }
    else dscale[i] = 1.0 / sqrt(gii);
}

__global__ void equil_scale_kernel(const double *__restrict__ G, const double *__restrict__ dscale,
                                   double *__restrict__ Lf, int n) {
    const long long id = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= (long long)n * n) return;
    const int r = (int)(id / n), c = (int)(id % n);
    Lf[id] = c <= r ? dscale[r] * G[id] * dscale[c] : 0.0;
}

constexpr int MP = 8;       // micro-panel width = the DMMA tile

__device__ __forceinline__ void dmma884(double &d0, double &d1, double a, double b);

// ---- panel step of the blocked Cholesky ------------------------------------------------------------------------
// One launch per 64-column panel; CTA b owns the 64 rows r0.. below the diagonal block and (redundantly, like every
// CTA of the launch) the diagonal block itself: a 128 x 64 matrix M = [A_kk; A_bk] in shared memory.  The panel is
// factored LEFT-LOOKING in micro-panels of 8 columns, the shape of the FP64 tensor instruction (mma.sync m8n8k4):
//   P/U(q) every 8-row tile t >= q of M:  M[t, Cq] -= M[t, C<q] M[q, C<q]^T           (DMMA, 2q k-steps)
//   D(q)   the warp that owns tile q factors the 8 x 8 diagonal tile IN REGISTERS (accumulator layout, columns
//          shared by shuffles: no barrier on the 8-pivot chain, rsqrt instead of sqrt and divide) and carries the
//          row operations along on an identity, which yields W = L_qq^-1 for free (micro_potrf)
//   S(q)   every tile t > q:  M[t, Cq] = M[t, Cq] W^T                                  (DMMA, 2 k-steps)
// so the rows below the diagonal -- of the diagonal block and of the panel alike -- never see a substitution chain,
// and the only serial work is D: the next owner solves and updates its own diagonal tile straight after barrier A
// and starts D(q + 1) while the other warps still work on step q (named barriers, bar.arrive for the owner).
// Measured on B200 (clock64 stamps, CTA 0 of panel 1, nothing else on the SM): D 1.35 k cycles, a step 1.8-2.0 k,
// the 8 steps 14-16 k, the whole panel 32 k cycles against 51 k for the round-1 kernel (one barrier per column
// across 256 threads, 445 cycles per column, then a 64-step shuffle substitution for the panel rows, bound by its
// shared-memory reads); with a science-side CTA on the same SM every phase takes 1.5-2 x longer.
// FUSED look-ahead (k0 > 0): the update of block column k0 by the previous panel (columns k0-64..k0-1) is applied on
// the way in: U_dd = X_d X_d^T and U_bd = X_b X_d^T (X_d, X_b: the previous panel's rows of the diagonal block and
// of this CTA's rows) by DMMA, subtracted from the tiles (which are loaded one phase ahead of their use) as they
// are written to M.  The trailing-update kernel then only covers block columns >= k0 + 64 and runs beside this
// kernel (launch_factor).
// CTA 0 writes L_kk to Ldiag, NOT back into Lf: the other CTAs of the launch read the unfactored block from Lf
// whenever they get scheduled.  grid = max(1, row tiles below); block 256; dynamic smem 2 * 64 * CLD doubles
// (X_d, X_b, then M) -- 70 KB, so a panel CTA fits beside a science-side CTA.

// acc = A B^T for two 64 x 64 shared-memory tiles (leading dimension CLD); 8 warps, warp tile 16 x 32: lane (fr, fk)
// holds rows rw + 8a + fr, columns cw + 8b + 2fk, +1 (the same fragment layout as syrk_kernel)
__device__ __forceinline__ void tile_abt(const double (*As)[CLD], const double (*Bs)[CLD], double (&acc)[2][4][2], int rw, int cw,
                                         int fr, int fk) {
#pragma unroll
    for (int a = 0; a < 2; a++)
#pragma unroll
        for (int b = 0; b < 4; b++) { acc[a][b][0] = 0.0; acc[a][b][1] = 0.0; }
#pragma unroll 4
    for (int kk = 0; kk < CB; kk += 4) {
        double af[2], bf[4];
#pragma unroll
        for (int a = 0; a < 2; a++) af[a] = As[rw + 8 * a + fr][kk + fk];
#pragma unroll
        for (int b = 0; b < 4; b++) bf[b] = Bs[cw + 8 * b + fr][kk + fk];
#pragma unroll
        for (int a = 0; a < 2; a++)
#pragma unroll
            for (int b = 0; b < 4; b++) dmma884(acc[a][b][0], acc[a][b][1], af[a], bf[b]);
    }
}

// D(q): Cholesky of the 8 x 8 diagonal tile and its inverse, by one warp, in the DMMA accumulator layout: lane
// (fr, fk) holds a[fr][2fk], a[fr][2fk+1] (lower triangle valid) and the same two entries of the row-reduced identity.
// Right-looking, all in registers: per column j four shuffles fetch the pivot, this row's a_rj and the two a_cj of
// this lane's columns (the tile is symmetric, so a_cj stands for a_jc), then a_rc -= a_rj a_cj / piv and
// L_rj = a_rj / sqrt(piv); the same row operations on an identity, u_r -= (l_rj / l_jj) u_j, give row j of
// W = L^-1 as u_j / l_jj at step j.  Column j of L and row j of W go to shared memory the moment they are final, so
// the updates run UNCONDITIONALLY afterwards (finished entries turn into finite garbage nobody reads): ~40
// instructions per column on a 119-cycle dependent chain (shuffle, rsqrt, two multiplies, fma).
__device__ __forceinline__ void micro_potrf(double a0, double a1, double (*M)[CLD], double (*Ws)[MP + 2], int q, int lane, int *flag,
                                            bool report) {
    const int fr = lane >> 2, fk = lane & 3;
    double w0 = (fr == 2 * fk) ? 1.0 : 0.0, w1 = (fr == 2 * fk + 1) ? 1.0 : 0.0;
    double *lrow = &M[MP * q + fr][MP * q];
    bool bad = false;
#pragma unroll
    for (int j = 0; j < MP; j++) {
        const int jh = j >> 1;
        const double aj = (j & 1) ? a1 : a0;                       // this lane's entry of column j if fk == jh
        double piv = __shfl_sync(0xffffffffu, aj, 4 * j + jh);
        const double arj = __shfl_sync(0xffffffffu, aj, (lane & ~3) | jh);
        const double ac0 = __shfl_sync(0xffffffffu, aj, 8 * fk + jh);
        const double ac1 = __shfl_sync(0xffffffffu, aj, 8 * fk + 4 + jh);
        const double uj0 = __shfl_sync(0xffffffffu, w0, 4 * j + fk);
        const double uj1 = __shfl_sync(0xffffffffu, w1, 4 * j + fk);
        if (!(piv > PIVOT_MIN)) { bad = true; piv = 1.0; }
        const double inv = rsqrt(piv);
        const double lrj = arj * inv;                              // row j: a_jj / sqrt(a_jj) = l_jj
        const double s = -lrj * inv;
        if (fk == jh) lrow[j] = lrj;                               // (rows above j store garbage right of the diagonal)
        if (fr == j) *reinterpret_cast<double2 *>(&Ws[j][2 * fk]) = make_double2(w0 * inv, w1 * inv);
        a0 = fma(s, ac0, a0); a1 = fma(s, ac1, a1);
        w0 = fma(s, uj0, w0); w1 = fma(s, uj1, w1);
    }
    if (bad && report && lane == 0) *flag = 1;
}

__global__ void __launch_bounds__(256, 2) potrf_panel_kernel(double *__restrict__ Lf, double *__restrict__ Ldiag, int n, int k0,
                                                             int bs, int *flag) {
    extern __shared__ __align__(16) double psm[];
    __shared__ __align__(16) double Ws[2][MP][MP + 2];
    double (*M)[CLD] = reinterpret_cast<double (*)[CLD]>(psm);   // rows 0..63: diagonal block, 64..127: this CTA's rows
    const int tid = threadIdx.x, lane = tid & 31, fr = lane >> 2, fk = lane & 3;
    // the warp index through a shuffle: the compiler then knows it is warp-uniform, and the shuffles and DMMA inside
    // the per-warp branches below compile without divergence guards (3 x fewer instructions in micro_potrf)
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
    const int rw = (warp >> 1) * 16, cw = (warp & 1) * 32;
    const int r0 = k0 + bs + blockIdx.x * CB;
    const bool have_rows = r0 < n;
    // the two tiles in the fragment layout of the products; every global load is issued one phase before its use:
    // the diagonal tile with the previous panel's rows, this CTA's tile before the second product
    double cur[2][4][2], acc[2][4][2];
#pragma unroll
    for (int a = 0; a < 2; a++)
#pragma unroll
        for (int b = 0; b < 4; b++)
#pragma unroll
            for (int h = 0; h < 2; h++) {
                const int r = rw + 8 * a + fr, c = cw + 8 * b + 2 * fk + h;
                double d = (r == c) ? 1.0 : 0.0;                   // identity padding for a short last block
                if (r < bs && c < bs) d = (c <= r) ? Lf[(size_t)(k0 + r) * n + k0 + c] : 0.0;
                cur[a][b][h] = d;
            }
    if (k0 > 0) {
        double (*Xd)[CLD] = reinterpret_cast<double (*)[CLD]>(psm);
        double (*Xb)[CLD] = reinterpret_cast<double (*)[CLD]>(psm + CB * CLD);
        const int kp = k0 - CB; // the previous panel is always a full block
        {
            double td[16], tb[16]; // all loads in flight before the first store (one global round trip, not sixteen)
#pragma unroll
            for (int i = 0; i < 16; i++) {
                const int e = tid + 256 * i, rr = e >> 6, cc = e & 63;
                td[i] = (k0 + rr < n) ? Lf[(size_t)(k0 + rr) * n + kp + cc] : 0.0;
                tb[i] = (have_rows && r0 + rr < n) ? Lf[(size_t)(r0 + rr) * n + kp + cc] : 0.0;
            }
#pragma unroll
            for (int i = 0; i < 16; i++) {
                const int e = tid + 256 * i, rr = e >> 6, cc = e & 63;
                Xd[rr][cc] = td[i]; Xb[rr][cc] = tb[i];
            }
        }
        __syncthreads();
        tile_abt(Xd, Xd, acc, rw, cw, fr, fk);
#pragma unroll
        for (int a = 0; a < 2; a++)
#pragma unroll
            for (int b = 0; b < 4; b++)
#pragma unroll
                for (int h = 0; h < 2; h++) {
                    const int r = rw + 8 * a + fr, c = cw + 8 * b + 2 * fk + h;
                    if (r < bs && c < bs && c <= r) cur[a][b][h] -= acc[a][b][h];
                }
    }
    double curb[2][4][2];
#pragma unroll
    for (int a = 0; a < 2; a++)
#pragma unroll
        for (int b = 0; b < 4; b++)
#pragma unroll
            for (int h = 0; h < 2; h++) {
                const int r = rw + 8 * a + fr, c = cw + 8 * b + 2 * fk + h;
                curb[a][b][h] = (have_rows && r0 + r < n && c < bs) ? Lf[(size_t)(r0 + r) * n + k0 + c] : 0.0;
            }
    if (k0 > 0) {
        double (*Xd)[CLD] = reinterpret_cast<double (*)[CLD]>(psm);
        double (*Xb)[CLD] = reinterpret_cast<double (*)[CLD]>(psm + CB * CLD);
        if (have_rows) {
            tile_abt(Xb, Xd, acc, rw, cw, fr, fk);
#pragma unroll
            for (int a = 0; a < 2; a++)
#pragma unroll
                for (int b = 0; b < 4; b++)
#pragma unroll
                    for (int h = 0; h < 2; h++) {
                        const int r = rw + 8 * a + fr, c = cw + 8 * b + 2 * fk + h;
                        if (r0 + r < n && c < bs) curb[a][b][h] -= acc[a][b][h];
                    }
        }
        __syncthreads();                                           // X_d, X_b are dead: M takes their place
    }
#pragma unroll
    for (int a = 0; a < 2; a++)
#pragma unroll
        for (int b = 0; b < 4; b++) {
            const int r = rw + 8 * a + fr, c = cw + 8 * b + 2 * fk;
            *reinterpret_cast<double2 *>(&M[r][c]) = make_double2(cur[a][b][0], cur[a][b][1]);
            *reinterpret_cast<double2 *>(&M[CB + r][c]) = make_double2(curb[a][b][0], curb[a][b][1]);
        }
    __syncthreads();
    // ---- the micro-panel pipeline -----------------------------------------------------------------------------
    // Warp w owns diagonal tile w and panel tile 8 + w (rows 64 + 8w..).  Step q:
    //   phase 1  warp q factors tile q (D); in its shadow the others apply the k-blocks < q to column block q + 1 (P)
    //   barrier A (everyone)
    //   phase 2  S(q): X = M[t, Cq] W^T.  Warp q + 1 does its diagonal tile only, ARRIVES at barrier B without
    //            waiting, applies the last k-block to that tile in registers and goes straight on to D(q + 1)
    //   barrier B (the others wait), phase 3: the last k-block q of column block q + 1 for all other tiles
    // so a step costs the chain D + A + four DMMA latencies.  The panel tile of a warp that is on the chain is handled
    // by the previous owner (which has no diagonal tile left).
    const bool rows = have_rows;
    constexpr int NQ = CB / MP;
    // M[t, cb] -= sum over k-blocks [p0, p1) of M[t, p] M[cb, p]^T; two accumulation chains
    auto upd = [&](int t, int cb, int p0, int p1) -> double2 {
        const double *ar = &M[MP * t + fr][fk], *br = &M[MP * cb + fr][fk];
        double2 c = *reinterpret_cast<const double2 *>(&M[MP * t + fr][MP * cb + 2 * fk]), e = make_double2(0.0, 0.0);
#pragma unroll 2
        for (int kk = MP * p0; kk < MP * p1; kk += 8) {
            dmma884(c.x, c.y, -ar[kk], br[kk]);
            dmma884(e.x, e.y, -ar[kk + 4], br[kk + 4]);
        }
        return make_double2(c.x + e.x, c.y + e.y);
    };
    auto put = [&](int t, int cb, double2 v) { *reinterpret_cast<double2 *>(&M[MP * t + fr][MP * cb + 2 * fk]) = v; };
    // X = M[t, Cq] W^T
    auto solve = [&](int t, int q, const double (*W)[MP + 2]) {
        const double w0 = W[fr][fk], w1 = W[fr][4 + fk];
        const double f0 = M[MP * t + fr][MP * q + fk], f1 = M[MP * t + fr][MP * q + 4 + fk];
        double2 x = make_double2(0.0, 0.0), y = x;
        dmma884(x.x, x.y, f0, w0);
        dmma884(y.x, y.y, f1, w1);
        __syncwarp();
        put(t, q, make_double2(x.x + y.x, x.y + y.y));
    };
    double2 dt = *reinterpret_cast<const double2 *>(&M[MP * warp + fr][MP * warp + 2 * fk]);   // used by warp 0 first
#pragma unroll 1
    for (int q = 0; q < NQ; q++) {
        const double (*W)[MP + 2] = Ws[q & 1];
        if (warp == q) micro_potrf(dt.x, dt.y, M, Ws[q & 1], q, lane, flag, blockIdx.x == 0);
        else if (q >= 1 && q + 1 < NQ) {
            if (warp > q) put(warp, q + 1, upd(warp, q + 1, 0, q));
            if (rows) {
                put(8 + warp, q + 1, upd(8 + warp, q + 1, 0, q));
                if (warp == q - 1) put(8 + q, q + 1, upd(8 + q, q + 1, 0, q));
            }
        }
        asm volatile("bar.sync 1, 256;" ::: "memory");             // A: W_q, L_qq and every P are in place
        if (warp == q + 1) {
            solve(warp, q, W);
            __syncwarp();
            asm volatile("bar.arrive 2, 256;" ::: "memory");       // B: X[q + 1, q] is out; do not wait for the others
            dt = upd(warp, q + 1, q, q + 1);
        } else {
            if (warp > q + 1) solve(warp, q, W);
            if (rows) {
                solve(8 + warp, q, W);
                if (warp == q && q + 1 < NQ) solve(8 + q + 1, q, W);
            }
            asm volatile("bar.sync 2, 256;" ::: "memory");         // B: every X[., q] is visible
            if (q + 1 < NQ) {
                if (warp > q + 1) put(warp, q + 1, upd(warp, q + 1, q, q + 1));
                if (rows) {
                    put(8 + warp, q + 1, upd(8 + warp, q + 1, q, q + 1));
                    if (warp == q) put(8 + q + 1, q + 1, upd(8 + q + 1, q + 1, q, q + 1));
                }
            }
        }
    }
    __syncthreads();
    // write-out, all shared-memory reads of a thread before its first store
    {
        const int c = tid & 63, rb = tid >> 6;
        if (blockIdx.x == 0) {
            double v[16];
#pragma unroll
            for (int i = 0; i < 16; i++) v[i] = M[rb + 4 * i][c];
#pragma unroll
            for (int i = 0; i < 16; i++) Ldiag[(rb + 4 * i) * CB + c] = c <= rb + 4 * i ? v[i] : 0.0;
        }
        if (have_rows) {
            double v[16];
#pragma unroll
            for (int i = 0; i < 16; i++) v[i] = M[CB + rb + 4 * i][c];
#pragma unroll
            for (int i = 0; i < 16; i++)
                if (r0 + rb + 4 * i < n && c < bs) Lf[(size_t)(r0 + rb + 4 * i) * n + k0 + c] = v[i];
        }
    }
}

// Inverses of the 64 x 64 diagonal blocks of the factor (identity-padded), for the triangular solves.
// Recursive: the four 16 x 16 diagonal sub-blocks are inverted in parallel by forward substitution (16 dependent
// steps instead of 64; thread (sub-block, column c, part) -- the 4 adjacent lanes of a column split every dot
// product), then the off-diagonal blocks follow from  X21 = -X22 (L21 X11)  at the 32 and the 64 level (two small
// products each, all 256 threads).  grid = number of blocks; block 256; dynamic smem 3 * 64 * 65 doubles.
__global__ void __launch_bounds__(256) trinv_kernel(double *__restrict__ Linv, int n, int blk0) {
    extern __shared__ __align__(16) double dsm[];
    double (*l)[CB + 1] = reinterpret_cast<double (*)[CB + 1]>(dsm);
    double (*x)[CB + 1] = reinterpret_cast<double (*)[CB + 1]>(dsm + CB * (CB + 1));
    double (*t)[CB + 1] = reinterpret_cast<double (*)[CB + 1]>(dsm + 2 * CB * (CB + 1));
    __shared__ double rdg[CB];
    // Linv[b] holds the factored diagonal block L_bb (identity-padded, written by potrf_panel_kernel): invert in place
    double *blk = Linv + (size_t)(blk0 + blockIdx.x) * CB * CB;
    const int tid = threadIdx.x;
    for (int e = tid; e < CB * CB; e += 256) { l[e >> 6][e & 63] = blk[e]; x[e >> 6][e & 63] = 0.0; }
    __syncthreads();
    if (tid < CB) rdg[tid] = 1.0 / l[tid][tid];
    __syncthreads();
    {   // 16 x 16 diagonal sub-blocks
        const int o = (tid >> 6) * 16, c = (tid >> 2) & 15, part = tid & 3;
        for (int i = 0; i < 16; i++) {
            double s = 0.0;
            for (int m = c + part; m < i; m += 4) s = fma(-l[o + i][o + m], x[o + m][o + c], s);
            s += __shfl_xor_sync(0xffffffffu, s, 1);
            s += __shfl_xor_sync(0xffffffffu, s, 2);
            if (part == 0) x[o + i][o + c] = i >= c ? ((i == c ? 1.0 : 0.0) + s) * rdg[o + i] : 0.0;
            __syncwarp();
        }
    }
    __syncthreads();
    // level 32: for h = 0, 1 the block rows o+16..o+31, columns o..o+15 (o = 32 h)
    {
        const int h = tid >> 7, o = 32 * h, e0 = tid & 127;
#pragma unroll
        for (int k = 0; k < 2; k++) { // T = L21 X11 (X11 lower triangular: m >= c)
            const int e = e0 + 128 * k, r = e >> 4, c = e & 15;
            double s = 0.0;
            for (int m = c; m < 16; m++) s = fma(l[o + 16 + r][o + m], x[o + m][o + c], s);
            t[o + 16 + r][o + c] = s;
        }
    }
    __syncthreads();
    {
        const int h = tid >> 7, o = 32 * h, e0 = tid & 127;
#pragma unroll
        for (int k = 0; k < 2; k++) { // X21 = -X22 T (X22 lower triangular: m <= r)
            const int e = e0 + 128 * k, r = e >> 4, c = e & 15;
            double s = 0.0;
            for (int m = 0; m <= r; m++) s = fma(-x[o + 16 + r][o + 16 + m], t[o + 16 + m][o + c], s);
            x[o + 16 + r][o + c] = s;
        }
    }
    __syncthreads();
    // level 64: rows 32..63, columns 0..31
#pragma unroll
    for (int k = 0; k < 4; k++) {
        const int e = tid + 256 * k, r = e >> 5, c = e & 31;
        double s = 0.0;
        for (int m = c; m < 32; m++) s = fma(l[32 + r][m], x[m][c], s);
        t[32 + r][c] = s;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < 4; k++) {
        const int e = tid + 256 * k, r = e >> 5, c = e & 31;
        double s = 0.0;
        for (int m = 0; m <= r; m++) s = fma(-x[32 + r][32 + m], t[32 + m][c], s);
        x[32 + r][c] = s;
    }
    __syncthreads();
    for (int e = tid; e < CB * CB; e += 256) blk[e] = x[e >> 6][e & 63];
}

__device__ __forceinline__ void dmma884(double &d0, double &d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

// trailing update: for block rows bi >= bj > kb:  A[bi][bj] -= X_bi X_bj^T,  X = panel columns k0..k0+bs.
// grid = ntile*(ntile+1)/2 lower-triangular tile pairs; block 256 = 8 warps, warp tile 16 x 32.
// mode 0: all tiles; 1: only the first block column (bj = 0; grid = ntile) -- all the next panel needs;
// 2: the other block columns (bj >= 1; grid = (ntile-1) ntile/2), run beside the next panel (look-ahead).
__global__ void __launch_bounds__(256) syrk_kernel(double *__restrict__ Lf, int n, int k0, int bs, int t0 /*first trailing row*/,
                                                  int mode) {
    extern __shared__ __align__(16) double dsm[];
    double (*As)[CLD] = reinterpret_cast<double (*)[CLD]>(dsm);
    double (*Bs)[CLD] = reinterpret_cast<double (*)[CLD]>(dsm + CB * CLD);
    // linear index -> (bi, bj), bj <= bi
    int idx = blockIdx.x, bi = 0, bj;
    if (mode == 1) { bi = idx; bj = 0; }
    else {
        while (idx > bi) { idx -= bi + 1; bi++; }
        bj = idx;
        if (mode == 2) { bi++; bj++; }
    }
    const int i0 = t0 + bi * CB, j0 = t0 + bj * CB;
    {   // all 32 loads of a thread in flight before the first shared-memory store: one global round trip, not sixteen
        double ta[16], tb[16];
#pragma unroll
        for (int i = 0; i < 16; i++) {
            const int e = threadIdx.x + 256 * i, r = e >> 6, c = e & 63;
            ta[i] = (i0 + r < n && c < bs) ? Lf[(size_t)(i0 + r) * n + k0 + c] : 0.0;
            tb[i] = (j0 + r < n && c < bs) ? Lf[(size_t)(j0 + r) * n + k0 + c] : 0.0;
        }
#pragma unroll
        for (int i = 0; i < 16; i++) {
            const int e = threadIdx.x + 256 * i, r = e >> 6, c = e & 63;
            As[r][c] = ta[i]; Bs[r][c] = tb[i];
        }
    }
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int rw = (warp >> 1) * 16, cw = (warp & 1) * 32;
    const int fr = lane >> 2, fk = lane & 3;
    double acc[2][4][2];
#pragma unroll
    for (int a = 0; a < 2; a++)
#pragma unroll
        for (int b = 0; b < 4; b++) { acc[a][b][0] = 0.0; acc[a][b][1] = 0.0; }
#pragma unroll 4
    for (int kk = 0; kk < CB; kk += 4) {
        double af[2], bf[4];
#pragma unroll
        for (int a = 0; a < 2; a++) af[a] = As[rw + 8 * a + fr][kk + fk];
#pragma unroll
        for (int b = 0; b < 4; b++) bf[b] = Bs[cw + 8 * b + fr][kk + fk];
#pragma unroll
        for (int a = 0; a < 2; a++)
#pragma unroll
            for (int b = 0; b < 4; b++) dmma884(acc[a][b][0], acc[a][b][1], af[a], bf[b]);
    }
    // read-modify-write of the 64 x 64 target tile: all reads first (the compiler must otherwise order each load behind
    // the previous store to the same array), then the stores
    double cur[2][4][2];
#pragma unroll
    for (int a = 0; a < 2; a++)
#pragma unroll
        for (int b = 0; b < 4; b++) {
            const int r = i0 + rw + 8 * a + fr, c = j0 + cw + 8 * b + 2 * fk;
            cur[a][b][0] = (r < n && c < n && c <= r) ? Lf[(size_t)r * n + c] : 0.0;
            cur[a][b][1] = (r < n && c + 1 < n && c + 1 <= r) ? Lf[(size_t)r * n + c + 1] : 0.0;
        }
#pragma unroll
    for (int a = 0; a < 2; a++)
#pragma unroll
        for (int b = 0; b < 4; b++) {
            const int r = i0 + rw + 8 * a + fr, c = j0 + cw + 8 * b + 2 * fk;
            if (r < n) {
                if (c < n && c <= r) Lf[(size_t)r * n + c] = cur[a][b][0] - acc[a][b][0];
                if (c + 1 < n && c + 1 <= r) Lf[(size_t)r * n + c + 1] = cur[a][b][1] - acc[a][b][1];
            }
        }
}

// ---- triangular solves: one CTA per 64-row block, all co-resident (cooperative launch) -------------
// c = D L^-T L^-1 D h.  Forward: CTA b accumulates L[b, kb] y_kb for kb = 0..b-1 as soon as block kb
// publishes y_kb, then solves its diagonal block and publishes y_b; backward the same from the last block up
// with L^T.  The critical path is the chain of 64 x 64 diagonal solves; the off-diagonal products of the
// waiting CTAs run beside it.
// Inter-CTA exchange of the solution blocks in the style of a low-latency flag-in-data protocol: a double travels as two
// 8-byte words (low half | epoch << 32), (high half | epoch << 32).  8-byte stores are atomic, so a reader that finds the
// epoch of THIS solve in both words has the value: one L2 round trip per hop instead of flag poll + fence + data load
// (the chain of 2 * nblk hops is the whole cost of the solve).  The epoch increments per call, so stale words never match.
// A reader gives up after ~1e6 polls and raises *err (a lost block must not hang the device).
__device__ __forceinline__ void ll_store(unsigned long long *buf, int i, double v, int epoch) {
    const unsigned long long b = (unsigned long long)__double_as_longlong(v), e = (unsigned long long)(unsigned)epoch << 32;
    volatile unsigned long long *w = buf + 2 * (size_t)i;
    w[0] = (b & 0xffffffffull) | e;
    w[1] = (b >> 32) | e;
}
__device__ __forceinline__ double ll_load(const unsigned long long *buf, int i, int epoch, int *err) {
    const volatile unsigned long long *w = buf + 2 * (size_t)i;
    const unsigned long long e = (unsigned long long)(unsigned)epoch;
    unsigned long long a = w[0], b = w[1];
    int spins = 0;
    while ((a >> 32) != e || (b >> 32) != e) {
        if (++spins > (1 << 20)) { *err = 3; return __longlong_as_double(0x7ff8000000000000LL); } // poison: a lost block must not yield plausible coefficients
        a = w[0]; b = w[1];
    }
    return __longlong_as_double((long long)((a & 0xffffffffull) | (b << 32)));
}

__global__ void __launch_bounds__(256) trisolve_kernel(const double *__restrict__ Lf, const double *__restrict__ Linv,
                                                      const double *__restrict__ dscale,
                                                      const double *__restrict__ h, unsigned long long *yl,
                                                      unsigned long long *zl, double *__restrict__ c, int n,
                                                      int *err, int epoch) {
    __shared__ double Ld[CB][CB + 1];
    __shared__ double vec[CB];
    __shared__ double blk[CB];
    __shared__ double part[4][CB];
    const int b = blockIdx.x, nblk = gridDim.x;
    const int k0 = b * CB, bs = min(CB, n - k0);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    for (int e = tid; e < CB * CB; e += 256) Ld[e >> 6][e & 63] = Linv[(size_t)b * CB * CB + e]; // inverse of L_bb
    // ---------------- forward: rows of this block, 8 rows per warp, lanes over the 64 columns of block kb
    // (everything the chain does not produce is fetched BEFORE the waits: a global load behind the arrival of y_{b-1}
    //  or z_{b+1} cost every hop of the chain a memory latency -- 3.3 us per forward hop, 1.5 us per backward hop)
    double rhs[8];
#pragma unroll
    for (int q = 0; q < 8; q++) { const int r = warp * 8 + q; rhs[q] = r < bs ? dscale[k0 + r] * h[k0 + r] : 0.0; }
    const double dsc_out = (tid >> 2) < bs ? dscale[k0 + (tid >> 2)] : 0.0;
    double acc[8];
#pragma unroll
    for (int q = 0; q < 8; q++) acc[q] = 0.0;
    for (int kb = 0; kb < b; kb++) {
        double l0[8], l1[8];
#pragma unroll
        for (int q = 0; q < 8; q++) { // L is final: load before waiting for y_kb
            const int r = warp * 8 + q;
            const double *row = Lf + (size_t)(k0 + r) * n + kb * CB;
            l0[q] = r < bs ? row[lane] : 0.0; l1[q] = r < bs ? row[lane + 32] : 0.0;
        }
        const double y0 = ll_load(yl, kb * CB + lane, epoch, err), y1 = ll_load(yl, kb * CB + lane + 32, epoch, err);
#pragma unroll
        for (int q = 0; q < 8; q++) acc[q] = fma(l0[q], y0, fma(l1[q], y1, acc[q]));
    }
#pragma unroll
    for (int q = 0; q < 8; q++) {
        double s = acc[q];
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) s += __shfl_down_sync(0xffffffffu, s, off);
        const int r = warp * 8 + q;
        if (lane == 0) blk[r] = r < bs ? rhs[q] - s : 0.0;
    }
    __syncthreads();
    {   // y_b = Linv_b * rhs: thread (r = tid/4, cq = tid%4) sums the columns c = cq mod 4
        const int r = tid >> 2, cq = tid & 3;
        double t = 0.0;
#pragma unroll
        for (int q = 0; q < 16; q++) t = fma(Ld[r][4 * q + cq], blk[4 * q + cq], t);
        t += __shfl_xor_sync(0xffffffffu, t, 1);
        t += __shfl_xor_sync(0xffffffffu, t, 2);
        __syncthreads();
        if (cq == 0) { blk[r] = t; ll_store(yl, k0 + r, r < bs ? t : 0.0, epoch); } // all 64 rows: readers take whole blocks
        __syncthreads();
    }
    // ---------------- backward: columns of this block; thread -> (col = tid % 64, slice = tid / 64)
    const int col = tid & (CB - 1), slice = tid >> 6;
    double s = 0.0;
    for (int kb = nblk - 1; kb > b; kb--) {
        const int i0 = kb * CB, ibs = min(CB, n - i0);
        double lv[16];
#pragma unroll
        for (int q = 0; q < 16; q++) {
            const int i = slice + 4 * q;
            lv[q] = (i < ibs && col < bs) ? Lf[(size_t)(i0 + i) * n + k0 + col] : 0.0;
        }
        if (tid < CB) vec[tid] = tid < ibs ? ll_load(zl, i0 + tid, epoch, err) : 0.0;
        __syncthreads();
#pragma unroll
        for (int q = 0; q < 16; q++) s = fma(lv[q], vec[slice + 4 * q], s);
        __syncthreads();
    }
    part[slice][col] = s;
    __syncthreads();
    if (tid < CB) blk[tid] = blk[tid] - (part[0][tid] + part[1][tid] + part[2][tid] + part[3][tid]);
    __syncthreads();
    {   // z_b = Linv_b^T * rhs
        const int cc = tid >> 2, cq = tid & 3;
        double t = 0.0;
#pragma unroll
        for (int q = 0; q < 16; q++) t = fma(Ld[4 * q + cq][cc], blk[4 * q + cq], t);
        t += __shfl_xor_sync(0xffffffffu, t, 1);
        t += __shfl_xor_sync(0xffffffffu, t, 2);
        if (cq == 0) {
            ll_store(zl, k0 + cc, cc < bs ? t : 0.0, epoch);   // the chain first, the output after it
            if (cc < bs) c[k0 + cc] = t * dsc_out;
        }
    }
}

cudaError_t launch_factor(sfft_plan *p) {
    const int n = p->g.n;
    cudaStream_t st = p->cur;
    if (!p->lf_ready) {   // (the gather of G normally leaves the equilibrated matrix behind: sfft_assemble.cu)
        cudaMemsetAsync(p->flag, 0, sizeof(int), st);
        { KLaunch kl(p, "equil_diag"); equil_diag_kernel<<<(n + 255) / 256, 256, 0, st>>>(p->G, p->dscale, n, p->flag); }
        const long long total = (long long)n * n;
        { KLaunch kl(p, "equil_scale"); equil_scale_kernel<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(p->G, p->dscale, p->Lf, n); }
    }
    p->lf_ready = false;  // the factor overwrites Lf
    const int nblk = (n + CB - 1) / CB;
    const size_t sm_syrk = 2 * CB * CLD * sizeof(double);
    cudaFuncSetAttribute(syrk_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm_syrk);
    cudaFuncSetAttribute(trinv_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(3 * CB * (CB + 1) * sizeof(double)));
    // Look-ahead: panel k+1 needs only the first block column of panel k's trailing update.  That part is fused into
    // the panel kernel of k+1; the rest of the update runs on an auxiliary stream beside it.
    cudaStream_t aux = (p->ktiming || !p->fstream2 || p->knob.no_lookahead) ? nullptr : p->fstream2;
    bool aux_busy = false;
    const size_t sm_panel = 2 * CB * CLD * sizeof(double);
    cudaFuncSetAttribute(potrf_panel_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm_panel);
    for (int kb = 0; kb < nblk; kb++) {
        const int k0 = kb * CB, bs = n - k0 < CB ? n - k0 : CB;
        const int rem = n - k0 - bs, nt = (rem + CB - 1) / CB;
        // panel kb, with the update of its block column by panel kb-1 fused in (potrf_panel_kernel).  It reads tiles the
        // rest-update of panel kb-2 (auxiliary stream) also wrote: the wait for that update was enqueued in iteration kb-1.
        { KLaunch kl(p, "potrf_panel"); potrf_panel_kernel<<<nt > 0 ? nt : 1, 256, sm_panel, st>>>(p->Lf, p->Linv + (size_t)kb * CB * CB, n, k0, bs, p->flag); }
        if (rem <= 0) continue;
        if (aux_busy) cudaStreamWaitEvent(st, p->ev_lookB, 0);              // panel kb+1 needs the rest-update of panel kb-1
        if (nt < 2) continue;                   // a single block column left: its update is the next panel's fused prologue
        // rest of the trailing update (block columns >= kb+2): beside the next panel kernel, whose 64-step dependent
        // chain leaves the machine almost empty
        if (!aux) {
            KLaunch kl(p, "syrk"); syrk_kernel<<<(nt - 1) * nt / 2, 256, sm_syrk, st>>>(p->Lf, n, k0, bs, k0 + bs, 2);
            continue;
        }
        cudaEventRecord(p->ev_lookP, st);                                   // panel kb is in place
        cudaStreamWaitEvent(aux, p->ev_lookP, 0);
        syrk_kernel<<<(nt - 1) * nt / 2, 256, sm_syrk, aux>>>(p->Lf, n, k0, bs, k0 + bs, 2);
        p->launches++;
        cudaEventRecord(p->ev_lookB, aux);
        aux_busy = true;
    }
    if (aux_busy) cudaStreamWaitEvent(st, p->ev_lookB, 0);
    // (inverting block kb on the auxiliary stream right after its panel delayed the look-ahead updates queued behind it)
    { KLaunch kl(p, "trinv"); trinv_kernel<<<nblk, 256, 3 * CB * (CB + 1) * sizeof(double), st>>>(p->Linv, n, 0); }
    cudaMemcpyAsync(p->flag_host, p->flag, sizeof(int), cudaMemcpyDeviceToHost, st);
    return cudaGetLastError();
}

cudaError_t launch_trisolve(sfft_plan *p, const double *h, double *c, cudaStream_t st, double *work) {
    const int n = p->g.n, nblk = (n + CB - 1) / CB;
    const double *Lf = p->Lf, *Li = p->Linv, *ds = p->dscale;
    p->solve_epoch++;
    const size_t wsz = 2 * (size_t)(((n + 63) / 64) * 64); // exchange words of one substitution (sfft_plan_create)
    unsigned long long *y = reinterpret_cast<unsigned long long *>(work ? work : p->ywork), *z = reinterpret_cast<unsigned long long *>(work ? work + wsz : p->zwork);
    int *err = p->flag + 1, epoch = p->solve_epoch, nn = n; // flag[0]: pivot test of the factorisation, flag[1]: solve errors
    void *args[] = {(void *)&Lf, (void *)&Li, (void *)&ds, (void *)&h, (void *)&y, (void *)&z, (void *)&c, (void *)&nn, (void *)&err, (void *)&epoch};
    KLaunch kl(p, "trisolve");
    return cudaLaunchCooperativeKernel((const void *)trisolve_kernel, dim3(nblk), dim3(256), args, 0, st ? st : p->stream);
}

// ---- sfft_solve_static: the same solve with its scratch in a file-scope device array (include/sfft.h) -----------
// Layout of the array, in doubles (every part starts on a 256-byte boundary):
//   Lf [MAX_N * MAX_N] (used with leading dimension n) | Linv [MAX_N / 64 blocks of 64 x 64] | dscale [MAX_N]
//   | y, z exchange words [2 * MAX_N each] | flags (2 ints: pivot test, solve error)
constexpr int SS_MAXN = SFFT_SOLVE_STATIC_MAX_N;
static_assert(SS_MAXN % CB == 0, "the scratch layout assumes whole blocks");
constexpr size_t SS_LF = 0, SS_LINV = SS_LF + (size_t)SS_MAXN * SS_MAXN, SS_DSC = SS_LINV + (size_t)SS_MAXN * CB,
                 SS_Y = SS_DSC + SS_MAXN, SS_Z = SS_Y + 2 * SS_MAXN, SS_FLAG = SS_Z + 2 * SS_MAXN, SS_TOTAL = SS_FLAG + 32;
static __device__ __align__(256) double g_solve_scratch[SS_TOTAL];

constexpr int SS_MAXDEV = 64;
struct StaticSolveDev { double *base; int epoch; };
static StaticSolveDev g_ss_dev[SS_MAXDEV];          // per device: the array's DEVICE address and the solve epoch
static std::mutex g_ss_mutex;
static thread_local char g_ss_err[256];

static sfft_status ss_fail(sfft_status st, const char *fmt, ...) {
    va_list ap; va_start(ap, fmt); vsnprintf(g_ss_err, sizeof g_ss_err, fmt, ap); va_end(ap);
    return st;
}

// Once per device, with that device current.  In host code the name g_solve_scratch is a host-side stand-in, not a
// device address: the kernels get the address cudaGetSymbolAddress returns for THIS device.
static cudaError_t ss_setup(int dev, cudaStream_t st, StaticSolveDev **out) {
    std::lock_guard<std::mutex> lock(g_ss_mutex);
    StaticSolveDev &d = g_ss_dev[dev];
    if (!d.base) {
        double *ptr = nullptr;
        cudaError_t e = cudaGetSymbolAddress((void **)&ptr, g_solve_scratch);
        if (e != cudaSuccess) return e;
        if (!ptr) return cudaErrorInvalidSymbol;
        // epoch 0 never matches a solve: the exchange words start cleared
        e = cudaMemsetAsync(ptr + SS_Y, 0, sizeof(double) * 4 * SS_MAXN, st);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(syrk_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(2 * CB * CLD * sizeof(double)));
        if (e == cudaSuccess) e = cudaFuncSetAttribute(potrf_panel_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(2 * CB * CLD * sizeof(double)));
        if (e == cudaSuccess) e = cudaFuncSetAttribute(trinv_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(3 * CB * (CB + 1) * sizeof(double)));
        if (e != cudaSuccess) return e;
        d.base = ptr; d.epoch = 0;
    }
    if (d.epoch == 0x7fffffff) {                   // the epoch is about to repeat: start over from cleared words
        const cudaError_t e = cudaMemsetAsync(d.base + SS_Y, 0, sizeof(double) * 4 * SS_MAXN, st);
        if (e != cudaSuccess) return e;
        d.epoch = 0;
    }
    d.epoch++;
    *out = &d;
    return cudaSuccess;
}

} // namespace sfft

extern "C" const char *sfft_solve_static_last_error(void) { return sfft::g_ss_err; }

extern "C" sfft_status sfft_solve_static(const double *G, const double *h, double *c, int n, void *cuda_stream) {
    using namespace sfft;
    g_ss_err[0] = 0;
    if (!G || !h || !c) return ss_fail(SFFT_ERR_INVALID_ARG, "sfft_solve_static: NULL pointer");
    if (n < 1 || n > SS_MAXN)
        return ss_fail(SFFT_ERR_INVALID_ARG, "sfft_solve_static: n = %d is outside 1..%d (SFFT_SOLVE_STATIC_MAX_N, the size of the static scratch array)", n, SS_MAXN);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return ss_fail(SFFT_ERR_CUDA, "sfft_solve_static: cudaGetDevice: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= SS_MAXDEV) return ss_fail(SFFT_ERR_INVALID_ARG, "sfft_solve_static: device %d not supported (< %d)", dev, SS_MAXDEV);
    StaticSolveDev *d = nullptr;
    e = ss_setup(dev, st, &d);
    if (e != cudaSuccess) return ss_fail(SFFT_ERR_CUDA, "sfft_solve_static: set-up: %s", cudaGetErrorString(e));
    double *Lf = d->base + SS_LF, *Linv = d->base + SS_LINV, *dscale = d->base + SS_DSC;
    unsigned long long *y = reinterpret_cast<unsigned long long *>(d->base + SS_Y), *z = reinterpret_cast<unsigned long long *>(d->base + SS_Z);
    int *flag = reinterpret_cast<int *>(d->base + SS_FLAG);
    const int nblk = (n + CB - 1) / CB;
    const size_t sm_mm = 2 * CB * CLD * sizeof(double);
    cudaMemsetAsync(flag, 0, 2 * sizeof(int), st);  // the flags must start at zero; everything else is overwritten
    equil_diag_kernel<<<(n + 255) / 256, 256, 0, st>>>(G, dscale, n, flag);
    equil_scale_kernel<<<(unsigned)(((long long)n * n + 255) / 256), 256, 0, st>>>(G, dscale, Lf, n);
    for (int kb = 0; kb < nblk; kb++) {             // launch_factor's sequence on ONE stream (no look-ahead stream or events)
        const int k0 = kb * CB, bs = n - k0 < CB ? n - k0 : CB;
        const int rem = n - k0 - bs, nt = (rem + CB - 1) / CB;
        potrf_panel_kernel<<<nt > 0 ? nt : 1, 256, sm_mm, st>>>(Lf, Linv + (size_t)kb * CB * CB, n, k0, bs, flag);
        if (nt >= 2) syrk_kernel<<<(nt - 1) * nt / 2, 256, sm_mm, st>>>(Lf, n, k0, bs, k0 + bs, 2);
    }
    trinv_kernel<<<nblk, 256, 3 * CB * (CB + 1) * sizeof(double), st>>>(Linv, n, 0);
    {
        const double *cLf = Lf, *cLi = Linv, *cds = dscale;
        int *err = flag + 1, epoch = d->epoch, nn = n;
        void *args[] = {(void *)&cLf, (void *)&cLi, (void *)&cds, (void *)&h, (void *)&y, (void *)&z, (void *)&c, (void *)&nn, (void *)&err, (void *)&epoch};
        e = cudaLaunchCooperativeKernel((const void *)trisolve_kernel, dim3(nblk), dim3(256), args, 0, st);
        if (e != cudaSuccess) return ss_fail(SFFT_ERR_CUDA, "sfft_solve_static: trisolve launch: %s", cudaGetErrorString(e));
    }
    int hf[2] = {0, 0};
    e = cudaMemcpyAsync(hf, flag, sizeof hf, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e != cudaSuccess) return ss_fail(SFFT_ERR_CUDA, "sfft_solve_static: %s", cudaGetErrorString(e));
    if (hf[0]) return ss_fail(SFFT_ERR_NOT_SPD, "sfft_solve_static: a pivot of the equilibrated matrix was <= 1e-12 (or a diagonal entry <= 0)");
    if (hf[1]) return ss_fail(SFFT_ERR_CUDA, "sfft_solve_static: a triangular-solve block never arrived; c is NaN");
    return SFFT_OK;
}
