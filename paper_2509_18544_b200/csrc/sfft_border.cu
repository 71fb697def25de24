// sfft_border.cu -- the native-grid wrap corrections of step a2 (reading C6: the method's sums are
// circular at nx x ny, the FFTs run on the zero-padded Mx x My grid).
//
// With lin = the part of a 1-D shifted sum whose shifted index stays inside the frame, wN / wM = the
// part that wraps on the native / padded grid (wM only where it lands on a real pixel again):
//   X_N = (lin_x + wN_x)(lin_y + wN_y),   X_M = (lin_x + wM_x)(lin_y + wM_y)
//   X_N - X_M = lin_x wN_y + wN_x lin_y + wN_x wN_y - lin_x wM_y - wM_x lin_y - wM_x wM_y .
// "lin_x wN_y" pairs one of the W rows at one end of the frame with one of the W rows at the other
// end and correlates them LINEARLY along x; "wN_x lin_y" does the same for column pairs along y; the
// last terms are |du| x |dv| corner sums.  So the correction is
//   strip_gather    the W first/last rows and columns of m.R (and m.S), columns transposed
//   linpair_kernel  linear 1-D correlations, all lags |e| <= W and coordinate powers, of every
//                   (line at one end, line at the other end) pair whose wrap distance is <= W
//   border_combine  per (pair, du, dv): the weighted sum of those plus the corner terms
// a few 1e8 multiply-adds in all (the bulk X_M comes from the spectra, sfft_lags.cu).
#include "sfft_internal.h"

namespace sfft {

__device__ __forceinline__ double bpw(double b, int e) { double r = 1.0; for (int k = 0; k < e; k++) r *= b; return r; }

// SB[img][side][k][pos], pos < NL.  side 0: row k;  1: row ny-1-k;  2: column k;  3: column nx-1-k.
// grid = (ceil(NL/256), W, 4*nimg); block 256.
__global__ void __launch_bounds__(256) strip_gather_kernel(const double *__restrict__ R, const double *__restrict__ S,
                                                          const uint8_t *__restrict__ mask, double *__restrict__ SB,
                                                          int W, int NL, int img0, Geom g) {
    const int pos = blockIdx.x * blockDim.x + threadIdx.x, k = blockIdx.y;
    const int img = img0 + blockIdx.z / 4, side = blockIdx.z & 3;
    const double *src = img == 0 ? R : S;
    const int n = side < 2 ? g.nx : g.ny;
    double v = 0.0;
    if (pos < n) {
        int x, y;
        if (side == 0) { x = pos; y = k; } else if (side == 1) { x = pos; y = g.ny - 1 - k; }
        else if (side == 2) { x = k; y = pos; } else { x = g.nx - 1 - k; y = pos; }
        const size_t o = (size_t)y * g.nx + x;
        v = src[o];
        if (mask && !mask[o]) v = 0.0;
    }
    if (pos < NL) SB[(((size_t)img * 4 + side) * W + k) * NL + pos] = v;
}

// LP[chunk][dt][rI][zI][e+W][ea][eb]: dt = 2*dirn + typ; dirn 0 = row pairs (along x), 1 = column pairs
// (along y); typ 0: a = high-end line rI (index n-1-rI), b = low-end line zI; typ 1: a = low-end line zI,
// b = high-end line rI.  Needed only when (rI+1) + zI <= W.
//   out[e][ea][eb] = sum_{pos in chunk, 0 <= pos+e < n} c(pos)^ea a[pos] * c(pos+e)^eb b[pos+e]
// grid = (nchunk, W*W, 4); block 256; dynamic smem (2*CH + 2W) doubles.
template <int EA, int EB>
__global__ void __launch_bounds__(256) linpair_kernel(const double *__restrict__ SBa, const double *__restrict__ SBb,
                                                     int W, int NL, int CH, double *__restrict__ LP, Geom g) {
    extern __shared__ __align__(16) double bsm[];
    const int rI = blockIdx.y / W, zI = blockIdx.y % W;
    if (rI + 1 + zI > W) return;
    const int dirn = blockIdx.z >> 1, typ = blockIdx.z & 1;
    const int n = dirn == 0 ? g.nx : g.ny;
    const double *hi = nullptr, *lo = nullptr;
    const double *a = SBa + ((size_t)(2 * dirn + (typ == 0 ? 1 : 0)) * W + (typ == 0 ? rI : zI)) * NL;
    const double *b = SBb + ((size_t)(2 * dirn + (typ == 0 ? 0 : 1)) * W + (typ == 0 ? zI : rI)) * NL;
    (void)hi; (void)lo;
    double *sa = bsm, *sb = bsm + CH;
    const int p0 = blockIdx.x * CH;
    for (int k = threadIdx.x; k < CH; k += blockDim.x) sa[k] = (p0 + k < n) ? a[p0 + k] : 0.0;
    for (int k = threadIdx.x; k < CH + 2 * W; k += blockDim.x) {
        const int p = p0 + k - W;
        sb[k] = (p >= 0 && p < n) ? b[p] : 0.0;
    }
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = blockDim.x >> 5;
    const double inv_n = 1.0 / (double)n;
    const size_t slot = ((((size_t)blockIdx.x * 4 + blockIdx.z) * W + rI) * W + zI) * (2 * W + 1);
    // c(pos + e) = c(pos) + delta, delta = 2e/n, so c(pos)^ea c(pos+e)^eb = sum_m C(eb, m) delta^(eb-m) c(pos)^(ea+m): the
    // EA x EB weighted correlations of a lag follow from the EA + EB - 1 moments M_k = sum_pos c(pos)^k a[pos] b[pos+e]
    // (7 running sums instead of 16 products for DK = 3, 5 instead of 9 for DK = 2: the kernel is FP64-bound).
    constexpr int NM = EA + EB - 1;
    for (int ei = warp; ei <= 2 * W; ei += nw) {
        const int e = ei - W;
        double mom[NM];
#pragma unroll
        for (int k = 0; k < NM; k++) mom[k] = 0.0;
        for (int k = lane; k < CH; k += 32) {
            const double ca = (2.0 * (p0 + k) + 1.0 - n) * inv_n;
            double t = sa[k] * sb[k + W + e];
#pragma unroll
            for (int m = 0; m < NM; m++) { mom[m] += t; t *= ca; }
        }
#pragma unroll
        for (int m = 0; m < NM; m++) {
            double v = mom[m];
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) v += __shfl_down_sync(0xffffffffu, v, off);
            mom[m] = v;
        }
        if (lane == 0) {
            const double delta = 2.0 * e * inv_n;
            double dp[EB];   // delta^j
            dp[0] = 1.0;
#pragma unroll
            for (int j = 1; j < EB; j++) dp[j] = dp[j - 1] * delta;
#pragma unroll
            for (int i = 0; i < EA; i++)
#pragma unroll
                for (int j = 0; j < EB; j++) {
                    double v = 0.0, binom = 1.0;   // C(j, m), m = 0..j
#pragma unroll
                    for (int m = 0; m <= j; m++) {
                        v = fma(binom * dp[j - m], mom[i + m], v);
                        binom = binom * (double)(j - m) / (double)(m + 1);
                    }
                    LP[((slot + ei) * EA + i) * EB + j] = v;
                }
        }
    }
}

// One WARP per (pair, du, dv): bpart[pair][dvIdx*(2W+1)+duIdx] = X_N - X_M (see the file header); the lanes
// share the wrapped rows, the wrapped columns and the corner terms, then reduce by shuffles.
__global__ void __launch_bounds__(128) border_combine_kernel(const double *__restrict__ LP, int nchunk, int W, int EA, int EB,
                                                            PairList pl, int sci, const double *__restrict__ R,
                                                            const double *__restrict__ S, const uint8_t *__restrict__ mask,
                                                            double *__restrict__ bpart, Geom g) {
    const int W2 = 2 * W + 1, nl = W2 * W2;
    const int id = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (id >= pl.np * nl) return;
    const int p = id / nl, lag = id - p * nl;
    const int du = lag % W2 - W, dv = lag / W2 - W;
    const int nx = g.nx, ny = g.ny;
    const int ia = g.pi[pl.a[p]], ja = g.pj[pl.a[p]];
    const int ib = sci ? 0 : g.pi[pl.b[p]], jb = sci ? 0 : g.pj[pl.b[p]];
    const double inx = 1.0 / nx, iny = 1.0 / ny;
    const size_t cstride = (size_t)4 * W * W * W2 * EA * EB; // one chunk of LP
    auto lp = [&](int dt, int rI, int zI, int ei, int ea, int eb) {
        const size_t o = (((((size_t)dt * W + rI) * W + zI) * W2 + ei) * EA + ea) * EB + eb;
        double s = 0.0;
        for (int c = 0; c < nchunk; c++) s += LP[c * cstride + o];
        return s;
    };
    auto cx = [&](int x) { return (2.0 * x + 1.0 - nx) * inx; };
    auto cy = [&](int y) { return (2.0 * y + 1.0 - ny) * iny; };
    double corr = 0.0;
    for (int pass = 0; pass < 2; pass++) { // 0: native-grid wraps (+), 1: padded-grid wraps that land on a pixel (-)
        const double sign = pass == 0 ? 1.0 : -1.0;
        const int ddx = abs(du) - (pass == 0 ? 0 : g.Mx - nx), ddy = abs(dv) - (pass == 0 ? 0 : g.My - ny);
        // rows wrap in y, x linear
        for (int k = lane; k < ddy; k += 32) {
            int r, z, ya, yb, typ;
            if (dv > 0) { r = k + 1; z = ddy - r; ya = ny - r; yb = z; typ = 0; }
            else { z = k; r = ddy - z; ya = z; yb = ny - r; typ = 1; }
            corr += sign * bpw(cy(ya), ja) * bpw(cy(yb), jb) * lp(typ, r - 1, z, du + W, ia, sci ? 0 : ib);
        }
        // columns wrap in x, y linear
        for (int k = lane; k < ddx; k += 32) {
            int r, z, xa, xb, typ;
            if (du > 0) { r = k + 1; z = ddx - r; xa = nx - r; xb = z; typ = 0; }
            else { z = k; r = ddx - z; xa = z; xb = nx - r; typ = 1; }
            corr += sign * bpw(cx(xa), ia) * bpw(cx(xb), ib) * lp(2 + typ, r - 1, z, dv + W, ja, sci ? 0 : jb);
        }
        // corners: both wrap
        const int ncorn = (ddx > 0 && ddy > 0) ? ddx * ddy : 0;
        for (int e = lane; e < ncorn; e += 32) {
            const int ky = e / ddx, kx = e - ky * ddx;
            int ya, yb, xa, xb;
            if (dv > 0) { ya = ny - (ky + 1); yb = ddy - (ky + 1); } else { ya = ky; yb = ny - (ddy - ky); }
            if (du > 0) { xa = nx - (kx + 1); xb = ddx - (kx + 1); } else { xa = kx; xb = nx - (ddx - kx); }
            const size_t oa = (size_t)ya * nx + xa, ob = (size_t)yb * nx + xb;
            double a = R[oa], b = sci ? S[ob] : R[ob];
            if (mask) { if (!mask[oa]) a = 0.0; if (!mask[ob]) b = 0.0; }
            corr += sign * (bpw(cx(xa), ia) * bpw(cy(ya), ja) * a) * (bpw(cx(xb), ib) * bpw(cy(yb), jb) * b);
        }
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) corr += __shfl_down_sync(0xffffffffu, corr, off);
    if (lane == 0) bpart[(size_t)p * nl + lag] = corr;
}

size_t border_lp_doubles(const Geom &g, int W, int EB) {
    return (size_t)border_linpair_chunks() * 4 * W * W * (2 * W + 1) * (g.DK + 1) * EB;
}
size_t border_strip_doubles(const Geom &g, int W) { return (size_t)2 * 4 * W * (g.nx > g.ny ? g.nx : g.ny); }
int border_linpair_chunks() { return 4; }

template <int EA, int EB>
static void run_linpair(sfft_plan *p, const double *SBa, const double *SBb, int W, int NL, int CH, int nchunk) {
    const size_t smem = (size_t)(2 * CH + 2 * W) * sizeof(double);
    linpair_kernel<EA, EB><<<dim3(nchunk, W * W, 4), 256, smem, p->cur>>>(SBa, SBb, W, NL, CH, p->LP, p->g);
}

// bpart[pair][(2W+1)^2] <- X_N - X_M for the pair list (science: b = m.S, else b = the template images)
cudaError_t launch_border(sfft_plan *p, const PairList &pl, int W, bool science, double *bpart) {
    const Geom &g = p->g;
    const int NL = g.nx > g.ny ? g.nx : g.ny, nchunk = border_linpair_chunks();
    const int CH = (NL + nchunk - 1) / nchunk;
    double *SB = p->SB; // [img][side][W][NL] with this call's W
    const size_t img_stride = (size_t)4 * W * NL;
    {
        KLaunch kl(p, science ? "strip_gather_S" : "strip_gather_R");
        // template strips are gathered with the template's W on the Omega call and again (narrower) on Theta calls
        strip_gather_kernel<<<dim3((NL + 255) / 256, W, science ? 8 : 4), 256, 0, p->cur>>>(p->R, p->S, p->mask, SB, W, NL, 0, g);
    }
    {
        KLaunch kl(p, science ? "linpair_theta" : "linpair_omega");
        const double *SBa = SB, *SBb = science ? SB + img_stride : SB;
        const int E = g.DK + 1;
        if (science) {
            if (E == 1) run_linpair<1, 1>(p, SBa, SBb, W, NL, CH, nchunk);
            else if (E == 2) run_linpair<2, 1>(p, SBa, SBb, W, NL, CH, nchunk);
            else if (E == 3) run_linpair<3, 1>(p, SBa, SBb, W, NL, CH, nchunk);
            else run_linpair<4, 1>(p, SBa, SBb, W, NL, CH, nchunk);
        } else {
            if (E == 1) run_linpair<1, 1>(p, SBa, SBb, W, NL, CH, nchunk);
            else if (E == 2) run_linpair<2, 2>(p, SBa, SBb, W, NL, CH, nchunk);
            else if (E == 3) run_linpair<3, 3>(p, SBa, SBb, W, NL, CH, nchunk);
            else run_linpair<4, 4>(p, SBa, SBb, W, NL, CH, nchunk);
        }
    }
    {
        KLaunch kl(p, science ? "border_combine_theta" : "border_combine_omega");
        const int total = pl.np * (2 * W + 1) * (2 * W + 1);
        border_combine_kernel<<<(total + 3) / 4, 128, 0, p->cur>>>(p->LP, nchunk, W, g.DK + 1, science ? 1 : g.DK + 1, pl,
                                                                            science ? 1 : 0, p->R, p->S, p->mask, bpart, g);
    }
    return cudaGetLastError();
}

} // namespace sfft
