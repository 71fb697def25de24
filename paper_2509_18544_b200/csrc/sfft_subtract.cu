// sfft_subtract.cu -- step a5 (BASELINE.json north_star (d)):
//   M = sum_t T_t (*) K_t  (circular at nx x ny, T_t = xt^i yt^j R UNMASKED, K_t[u,v] = a_{t,u,v}),
//   D = S - M - B,  B = sum_s b_s xt^p yt^q.
// By FFT on the zero-padded Mx x My grid:  M^ = sum_t T^_t K^_t,
//   K^_t[ky,kx] = sum_v e^{-2 pi i ky v/My} E_t[v][kx],  E_t[v][kx] = sum_u a_{t,u,v} e^{-2 pi i kx u/Mx}.
// Kernels:
//   ktab_plain, col_inv (sfft_cols.cu)  M^ column by column (K^ synthesised on the fly) + inverse FFT along y
//   row_inv (sfft_rows.cu)              Hermitian -> packed, inverse FFT along x, fused D = S - M - B
//   wrapfix_kernel (here)               pixels within w of the frame edge: replace the taps that wrap on the padded
//                                       grid by the taps that wrap on the native grid (reading C6)
#include "sfft_internal.h"

namespace sfft {

// One thread per border pixel (within w of an edge).  For every tap (u,v) whose source pixel
// (x-u, y-v) leaves the frame, the padded-grid FFT used Rpad((x-u) mod Mx, (y-v) mod My) (zero in
// the padding) where the method wants R((x-u) mod nx, (y-v) mod ny): subtract the difference.
// Two kernels: wrapcorr computes the corrections (they depend on R and the coefficients only, so it runs on a side stream
// BESIDE the inverse transforms) into corr[border pixel id]; wrapapply subtracts them from D afterwards.
__global__ void __launch_bounds__(128) wrapcorr_kernel(const double *__restrict__ R, const double *__restrict__ coef,
                                                      double *__restrict__ cbuf, Geom g) {
    const int nx = g.nx, ny = g.ny, w = g.w, L = g.L, LL = L * L;
    const long long nA = 2LL * w * nx, nB = 2LL * w * (ny - 2 * w);
    // 4 adjacent lanes share a pixel (tap rows v = -w + part, step 4): the per-thread chain of dependent R loads is 4x shorter
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int part = (int)(gid & 3);
    const bool live = (gid >> 2) < nA + nB;
    const long long id = live ? (gid >> 2) : 0;
    int x, y;
    if (id < nA) { const int r = (int)(id / nx); x = (int)(id - (long long)r * nx); y = r < w ? r : ny - 2 * w + r; }
    else { const long long k = id - nA; const int r = (int)(k / (2 * w)), cidx = (int)(k - (long long)r * 2 * w); y = w + r; x = cidx < w ? cidx : nx - 2 * w + cidx; }
    const double inx = 1.0 / nx, iny = 1.0 / ny;
    // taps whose source column leaves the frame: u in (x, w] (left edge) or u in [-w, x - nx] (right edge)
    const int ulo_in = max(-w, x - nx + 1), uhi_in = min(w, x); // u in [ulo_in, uhi_in] stays inside
    double corr = 0.0;
    // K(u,v; x',y') R(x',y') at a wrapped source pixel
    auto term = [&](int u, int v, int xs, int ys) {
        const double xt = (2.0 * xs + 1.0 - nx) * inx, yt = (2.0 * ys + 1.0 - ny) * iny;
        double xp[MAX_DEG + 1], yp[MAX_DEG + 1];
        xp[0] = 1.0; yp[0] = 1.0;
#pragma unroll
        for (int k = 1; k <= MAX_DEG; k++) { xp[k] = xp[k - 1] * xt; yp[k] = yp[k - 1] * yt; }
        const double *a = coef + (size_t)(v + w) * L + (u + w);
        double k = 0.0;
        int t = 0;
#pragma unroll
        for (int d = 0; d <= MAX_DEG; d++)
#pragma unroll
            for (int j = 0; j <= d; j++, t++)
                if (d <= g.DK) k = fma(a[(size_t)t * LL], xp[d - j] * yp[j], k);
        return k * R[(size_t)ys * nx + xs];
    };
    for (int v = -w + part; v <= w; v += 4) {
        const int ys = y - v;
        const bool oy = ys < 0 || ys >= ny;
        const int yN = ys < 0 ? ys + ny : (ys >= ny ? ys - ny : ys), yM = (ys + g.My) & (g.My - 1);
        for (int u = -w; u <= w; u++) {
            if (!oy && u >= ulo_in && u <= uhi_in) { u = uhi_in; continue; } // skip the in-frame run
            const int xs = x - u;
            const int xN = xs < 0 ? xs + nx : (xs >= nx ? xs - nx : xs), xM = (xs + g.Mx) & (g.Mx - 1);
            corr += term(u, v, xN, yN);                                  // native-grid wrap: + value
            if (xM < nx && yM < ny) corr -= term(u, v, xM, yM);          // padded-grid wrap landed on a real pixel
        }
    }
    corr += __shfl_xor_sync(0xffffffffu, corr, 1);
    corr += __shfl_xor_sync(0xffffffffu, corr, 2);
    if (live && part == 0) cbuf[id] = corr;
}

__global__ void __launch_bounds__(256) wrapapply_kernel(const double *__restrict__ cbuf, double *__restrict__ D, Geom g, int mode) {
    const int nx = g.nx, ny = g.ny, w = g.w;
    const long long nA = 2LL * w * nx, nB = 2LL * w * (ny - 2 * w);
    const long long id = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= nA + nB) return;
    int x, y;
    if (id < nA) { const int r = (int)(id / nx); x = (int)(id - (long long)r * nx); y = r < w ? r : ny - 2 * w + r; }
    else { const long long k = id - nA; const int r = (int)(k / (2 * w)), cidx = (int)(k - (long long)r * 2 * w); y = w + r; x = cidx < w ? cidx : nx - 2 * w + cidx; }
    const double c = cbuf[id];
    D[(size_t)y * nx + x] -= mode ? -c : c;
}

cudaError_t launch_subtract(sfft_plan *p, const double *S, const double *R, const double *coef, double *D,
                            const void *spec, int mode) {
    const Geom &g = p->g;
    if (!spec) spec = p->mask ? p->specTo : p->specT; // a mask keeps a second, unmasked set (C7); without one the fit spectra are it
    const bool fix = (g.Mx != g.nx || g.My != g.ny) && g.w > 0;
    const long long nb = 2LL * g.w * g.nx + 2LL * g.w * (g.ny - 2 * g.w);
    if (fix) {   // the corrections on a side stream beside the transforms (needs R and the coefficients only)
        fork_side(p);
        use_side(p, 0);
        { KLaunch kl(p, "wrapcorr"); wrapcorr_kernel<<<(unsigned)((4 * nb + 127) / 128), 128, 0, p->cur>>>(R, coef, p->wcorr, g); }
        back_to_main(p);
    }
    cudaError_t e = launch_col_inv(p, spec, coef, p->inter);
    if (e == cudaSuccess) e = launch_row_inv(p, p->inter, S, coef, D, mode);
    if (e != cudaSuccess) return e;
    if (fix) {
        join_side(p);
        KLaunch kl(p, "wrapapply");
        wrapapply_kernel<<<(unsigned)((nb + 255) / 256), 256, 0, p->stream>>>(p->wcorr, D, g, mode);
    }
    return cudaGetLastError();
}

} // namespace sfft
