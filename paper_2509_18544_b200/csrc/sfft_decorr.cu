// f1: the decorrelation kernel (pipeline step 7; readings D1-D5 of DESIGN.md section 13).
//   D = S (*) P_R - (R (*) P_S) (*) K - B  has the noise power spectrum
//       F(k) = var_S |P_R^(k)|^2 + var_R |P_S^(k)|^2 |K^(k)|^2            (white noise in S and R),
//   the decorrelation kernel is W^(k) = sqrt(F(0) / F(k)) on an N x N periodic grid, and what is applied to the
//   images (by sfft_convolve_stamp) is the central L x L crop of W.
// Everything here is a few thousand taps: the kernels are latency-bound set-up work (one call per frame), written as
// pruned direct DFTs -- only the P x P input taps are summed forward and only the L x L output taps are formed.
//   local_kernel_kernel   coefficients -> K(u, v; x, y) = sum_t a_{t,u,v} xt^i yt^j
//   decorr_power_kernel   the three stamps -> F[ky][kx] (one thread per frequency, exact integer phase reduction)
//   decorr_stamp_kernel   F -> stamp[v][u] = N^-2 sum_k sqrt(F(0)/F(k)) cos(2 pi (kx u + ky v)/N)  (one CTA per tap)
#include "sfft_internal.h"

namespace sfft {

// grid = ceil(L*L / 128), block 128
__global__ void local_kernel_kernel(const double *__restrict__ coef, double *__restrict__ K, Geom g, double xt, double yt) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x, LL = g.L * g.L;
    if (k >= LL) return;
    double acc = 0.0;
    for (int t = 0; t < g.NK; t++) {
        double wgt = 1.0;
        for (int e = 0; e < g.pi[t]; e++) wgt *= xt;
        for (int e = 0; e < g.pj[t]; e++) wgt *= yt;
        acc = fma(coef[(size_t)t * LL + k], wgt, acc);
    }
    K[k] = acc;
}

// sum_{u,v} st[(v+w) P + (u+w)] exp(-2 pi i (kx u + ky v)/N); the phase index is reduced mod N in integers
__device__ __forceinline__ cplx stamp_dft(const double *__restrict__ st, int P, int kx, int ky, int N) {
    const int w = (P - 1) / 2;
    const double s2 = 2.0 / (double)N;
    cplx z = mk(0, 0);
    for (int v = -w; v <= w; v++) {
        const int mv = (ky * (v + N)) % N;
        for (int u = -w; u <= w; u++) {
            const int m = (mv + kx * (u + N)) % N;
            double sn, cs;
            sincospi(s2 * (double)m, &sn, &cs);
            const double a = st[(v + w) * P + (u + w)];
            z.x = fma(a, cs, z.x); z.y = fma(-a, sn, z.y);
        }
    }
    return z;
}

// grid = ceil(N*N / 128), block 128.  bad: raised when F is not a positive finite number somewhere
__global__ void decorr_power_kernel(const double *__restrict__ K, int Lk, const double *__restrict__ PS,
                                    const double *__restrict__ PR, int Lp, double varS, double varR, int N,
                                    double *__restrict__ F, int *__restrict__ bad) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= N * N) return;
    const int ky = k / N, kx = k - ky * N;
    const cplx zk = stamp_dft(K, Lk, kx, ky, N), zs = stamp_dft(PS, Lp, kx, ky, N), zr = stamp_dft(PR, Lp, kx, ky, N);
    const double f = varS * (zr.x * zr.x + zr.y * zr.y) + varR * (zs.x * zs.x + zs.y * zs.y) * (zk.x * zk.x + zk.y * zk.y);
    F[k] = f;
    if (!(f > 0.0) || isinf(f)) atomicExch(bad, 1);
}

// grid = L*L (one CTA per output tap), block 256
__global__ void __launch_bounds__(256) decorr_stamp_kernel(const double *__restrict__ F, int N, int L,
                                                           double *__restrict__ stamp) {
    const int w = (L - 1) / 2, v = (int)blockIdx.x / L - w, u = (int)blockIdx.x % L - w;
    const double f0 = F[0], s2 = 2.0 / (double)N;
    double acc = 0.0;
    for (int k = threadIdx.x; k < N * N; k += blockDim.x) {
        const int ky = k / N, kx = k - ky * N;
        const int m = ((ky * (v + N)) % N + kx * (u + N)) % N;
        acc = fma(sqrt(f0 / F[k]), cospi(s2 * (double)m), acc);
    }
    __shared__ double part[8];
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int i = 0; i < 8; i++) s += part[i];
        stamp[blockIdx.x] = s / ((double)N * (double)N);
    }
}

cudaError_t launch_local_kernel(sfft_plan *p, const double *coef, double xt, double yt, double *K) {
    const int LL = p->g.L * p->g.L;
    KLaunch kl(p, "local_kernel");
    local_kernel_kernel<<<(LL + 127) / 128, 128, 0, p->stream>>>(coef, K, p->g, xt, yt);
    return cudaGetLastError();
}

cudaError_t launch_decorr(sfft_plan *p, const double *K, int Lk, const double *PS, const double *PR, int Lp,
                          double varS, double varR, int N, double *F, int *bad, double *stamp) {
    cudaError_t e = cudaMemsetAsync(bad, 0, sizeof(int), p->stream);
    if (e != cudaSuccess) return e;
    { KLaunch kl(p, "decorr_power"); decorr_power_kernel<<<(N * N + 127) / 128, 128, 0, p->stream>>>(K, Lk, PS, PR, Lp, varS, varR, N, F, bad); }
    { KLaunch kl(p, "decorr_stamp"); decorr_stamp_kernel<<<p->g.L * p->g.L, 256, 0, p->stream>>>(F, N, p->g.L, stamp); }
    return cudaGetLastError();
}

} // namespace sfft
