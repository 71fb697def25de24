// f3: alignment / resampling onto the science grid (pipeline step 4; readings A1-A4 of
// DESIGN.md section 14).  out(x, y) = interpolant of img at the affine source position
//     xs = (M0 x + M1 y) + M2,  ys = (M3 x + M4 y) + M5      (FP64, this order, no fused multiply-add: the integer
// decisions floor(xs), floor(xs + 0.5) and the footprint test are then the same bits as in the oracle).
// One thread per output pixel, 32 x 8 pixel CTAs: the 2a x 2a footprints of neighbouring pixels overlap, so the source
// is read from HBM once (through L1/L2: ncu 134 MB read at 4088^2); nearest and bilinear are bound by 1 r read + 1 r
// written, Lanczos-3 by the FP64 instructions of its 12 weights and 36 taps per pixel.
// With f = xs - floor(xs) and tap offsets k = -2..3:
//     sin(pi (f - k)) = (-1)^k sin(pi f),   sin(pi (f - k)/3) = sin(pi f/3) cos(k pi/3) - cos(pi f/3) sin(k pi/3).
#include "sfft_internal.h"

namespace sfft {

struct Affine { double m[6]; };

__device__ __forceinline__ void source_pos(const Affine &A, int x, int y, double &xs, double &ys) {
    xs = __dadd_rn(__dadd_rn(__dmul_rn(A.m[0], (double)x), __dmul_rn(A.m[1], (double)y)), A.m[2]);
    ys = __dadd_rn(__dadd_rn(__dmul_rn(A.m[3], (double)x), __dmul_rn(A.m[4], (double)y)), A.m[5]);
}

// Weights PROPORTIONAL to k(f - k), k = -2..3, k(t) = sinc(t) sinc(t/3): the caller divides by their sum (reading A2), so
// every factor common to the six taps is dropped -- 3/pi^2, |sin(pi f)| and 1/prod_j (f - j)^2:
//     w_k = (-1)^k sin(pi (f - k)/3) prod_{j != k} (f - j)^2.
// One sincospi and no division per axis (prefix / suffix products of the t^2); ncu shows the kernel bound by FP64
// instruction issue, not by HBM (profiles/r01o_align_ncu.md), so this is what its time is made of.
__device__ __forceinline__ void lanczos3_weights(double f, double w[6]) {
    const double H = 0.86602540378443864676372317075294;    // sqrt(3)/2
    const double ck[6] = {-0.5, 0.5, 1.0, 0.5, -0.5, -1.0}, sk[6] = {-H, -H, 0.0, H, H, 0.0};
    if (f == 0.0) { // on a pixel centre sin(pi f) = 0 kills every other tap (and the products below would all vanish)
#pragma unroll
        for (int q = 0; q < 6; q++) w[q] = q == 2 ? 1.0 : 0.0;
        return;
    }
    double s3, c3;
    sincospi(f * (1.0 / 3.0), &s3, &c3);
    double u[6], pre[6], suf[6];
#pragma unroll
    for (int q = 0; q < 6; q++) { const double t = f - (double)(q - 2); u[q] = t * t; }
    pre[0] = 1.0; suf[5] = 1.0;
#pragma unroll
    for (int q = 1; q < 6; q++) pre[q] = pre[q - 1] * u[q - 1];
#pragma unroll
    for (int q = 4; q >= 0; q--) suf[q] = suf[q + 1] * u[q + 1];
#pragma unroll
    for (int q = 0; q < 6; q++) {
        const double b = s3 * ck[q] - c3 * sk[q];     // sin(pi (f - k)/3)
        w[q] = ((q & 1) ? -b : b) * (pre[q] * suf[q]);
    }
}

template <int METHOD>
__global__ void __launch_bounds__(256) resample_kernel(const double *__restrict__ img, double *__restrict__ out,
                                                       int nx, int ny, Affine A, double fill) {
    const int x = blockIdx.x * 32 + threadIdx.x, y = blockIdx.y * 8 + threadIdx.y;
    if (x >= nx || y >= ny) return;
    double xs, ys;
    source_pos(A, x, y, xs, ys);
    double r = fill;
    if (METHOD == 0) {
        const double fx = floor(xs + 0.5), fy = floor(ys + 0.5);
        if (fx >= 0.0 && fx < (double)nx && fy >= 0.0 && fy < (double)ny) r = img[(size_t)(int)fy * nx + (int)fx];
    } else {
        constexpr int a = METHOD == 1 ? 1 : 3;
        const double fx = floor(xs), fy = floor(ys);
        if (fx - (a - 1) >= 0.0 && fx + a <= (double)(nx - 1) && fy - (a - 1) >= 0.0 && fy + a <= (double)(ny - 1)) {
            const int i0 = (int)fx, j0 = (int)fy;
            double wx[2 * a], wy[2 * a];
            if (METHOD == 1) {
                const double tx = xs - fx, ty = ys - fy;
                wx[0] = 1.0 - tx; wx[1] = 1.0 - fabs(xs - (fx + 1.0));
                wy[0] = 1.0 - ty; wy[1] = 1.0 - fabs(ys - (fy + 1.0));
            } else {
                lanczos3_weights(xs - fx, wx);
                lanczos3_weights(ys - fy, wy);
            }
            double sx = 0.0, sy = 0.0, acc = 0.0;
#pragma unroll
            for (int q = 0; q < 2 * a; q++) { sx += wx[q]; sy += wy[q]; }
#pragma unroll
            for (int qj = 0; qj < 2 * a; qj++) {
                const double *row = img + (size_t)(j0 - a + 1 + qj) * nx + (i0 - a + 1);
                double rs = 0.0;
#pragma unroll
                for (int qi = 0; qi < 2 * a; qi++) rs = fma(wx[qi], row[qi], rs);
                acc = fma(wy[qj], rs, acc);
            }
            r = acc / (sx * sy);
        }
    }
    out[(size_t)y * nx + x] = r;
}

__global__ void __launch_bounds__(256) resample_mask_kernel(const uint8_t *__restrict__ m, uint8_t *__restrict__ out,
                                                            int nx, int ny, Affine A, int fill) {
    const int x = blockIdx.x * 32 + threadIdx.x, y = blockIdx.y * 8 + threadIdx.y;
    if (x >= nx || y >= ny) return;
    double xs, ys;
    source_pos(A, x, y, xs, ys);
    const double fx = floor(xs + 0.5), fy = floor(ys + 0.5);
    uint8_t r = (uint8_t)fill;
    if (fx >= 0.0 && fx < (double)nx && fy >= 0.0 && fy < (double)ny) r = m[(size_t)(int)fy * nx + (int)fx];
    out[(size_t)y * nx + x] = r;
}

cudaError_t launch_resample(sfft_plan *p, const double *img, const double *M, int method, double fill, double *out) {
    const int nx = p->g.nx, ny = p->g.ny;
    Affine A;
    for (int i = 0; i < 6; i++) A.m[i] = M[i];
    const dim3 grid((nx + 31) / 32, (ny + 7) / 8), block(32, 8);
    KLaunch kl(p, "resample");
    if (method == 0) resample_kernel<0><<<grid, block, 0, p->stream>>>(img, out, nx, ny, A, fill);
    else if (method == 1) resample_kernel<1><<<grid, block, 0, p->stream>>>(img, out, nx, ny, A, fill);
    else resample_kernel<3><<<grid, block, 0, p->stream>>>(img, out, nx, ny, A, fill);
    return cudaGetLastError();
}

cudaError_t launch_resample_mask(sfft_plan *p, const uint8_t *mask, const double *M, int fill, uint8_t *out) {
    const int nx = p->g.nx, ny = p->g.ny;
    Affine A;
    for (int i = 0; i < 6; i++) A.m[i] = M[i];
    const dim3 grid((nx + 31) / 32, (ny + 7) / 8), block(32, 8);
    KLaunch kl(p, "resample_mask");
    resample_mask_kernel<<<grid, block, 0, p->stream>>>(mask, out, nx, ny, A, fill);
    return cudaGetLastError();
}

} // namespace sfft
