// f4 (first variant): the constant-photometric-ratio constraint (reading R1 of DESIGN.md section 15):
//     minimise |b - A c|^2  subject to  sum_{u,v} a_{t,u,v} = 0  for every polynomial term t = 1..NK-1.
// With the Cholesky factor of G already there (a4) this is a Schur-complement correction of the free solution c0 = G^-1 h:
//     z_k = G^-1 e_k  (e_k = indicator of the taps of term k; one more pair of triangular solves each),
//     Sm[k][k'] = e_k^T z_k',  r_k = e_k^T c0,  Sm lambda = r,  c = c0 - sum_k lambda_k z_k.
// Kernels: ratio_rhs_kernel writes the m = NK-1 indicator vectors; ratio_apply_kernel (one CTA) reduces Sm and r, solves
// the m x m system (m <= 9, symmetric positive definite: Gaussian elimination in one thread) and corrects c in place.
#include "sfft_internal.h"

namespace sfft {

// grid = (ceil(n/256), m)
__global__ void ratio_rhs_kernel(double *__restrict__ E, int n, int LL) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x, k = blockIdx.y + 1;
    if (i < n) E[(size_t)blockIdx.y * n + i] = (i >= k * LL && i < (k + 1) * LL) ? 1.0 : 0.0;
}

constexpr int RMAX = MAX_NP - 1;

// one CTA of 256 threads.  Z: [m][n] the solves z_k; c: [n] in/out
__global__ void __launch_bounds__(256) ratio_apply_kernel(const double *__restrict__ Z, double *__restrict__ c, int n,
                                                          int LL, int m) {
    __shared__ double Sm[RMAX][RMAX + 1]; // augmented with r
    __shared__ double lam[RMAX];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // entry (k, k') with k' = m meaning r_k: one warp per entry, strided over the LL taps of block k+1
    for (int e = warp; e < m * (m + 1); e += 8) {
        const int k = e / (m + 1), kp = e % (m + 1);
        const double *v = kp < m ? Z + (size_t)kp * n : c;
        double s = 0.0;
        for (int i = lane; i < LL; i += 32) s += v[(size_t)(k + 1) * LL + i];
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
        if (lane == 0) Sm[k][kp] = s;
    }
    __syncthreads();
    if (tid == 0) {
        for (int j = 0; j < m; j++) {           // elimination with partial pivoting on the augmented matrix
            int piv = j;
            for (int i = j + 1; i < m; i++) if (fabs(Sm[i][j]) > fabs(Sm[piv][j])) piv = i;
            if (piv != j) for (int q = 0; q <= m; q++) { const double t = Sm[j][q]; Sm[j][q] = Sm[piv][q]; Sm[piv][q] = t; }
            const double d = 1.0 / Sm[j][j];
            for (int i = j + 1; i < m; i++) {
                const double f = Sm[i][j] * d;
                for (int q = j; q <= m; q++) Sm[i][q] -= f * Sm[j][q];
            }
        }
        for (int j = m - 1; j >= 0; j--) {
            double s = Sm[j][m];
            for (int q = j + 1; q < m; q++) s -= Sm[j][q] * lam[q];
            lam[j] = s / Sm[j][j];
        }
    }
    __syncthreads();
    for (int i = tid; i < n; i += 256) {
        double v = c[i];
        for (int k = 0; k < m; k++) v -= lam[k] * Z[(size_t)k * n + i];
        c[i] = v;
    }
}

// E, Z: [m][n] each (plan-owned).  z_k = G^-1 e_k on stream st: they depend on the factor only, so the caller runs them
// right behind the factorisation (beside the science-side kernels) and keeps them for as long as the factor lives.
// The m solves are independent: solve 0 stays on st with the plan's exchange words, solves 1..m-1 run beside it on the
// plan's auxiliary streams with exchange words of their own (W; each is a 12-CTA latency chain, so five in parallel take
// about as long as one).  In per-launch timing mode everything stays on st.
cudaError_t launch_ratio_Z(sfft_plan *p, double *E, double *Z, cudaStream_t st, double *W) {
    const int n = p->g.n, LL = p->g.L * p->g.L, m = p->g.NK - 1;
    if (m < 1) return cudaSuccess;
    const size_t wsz = 2 * (size_t)(((n + 63) / 64) * 64);
    const bool par = W && !p->ktiming && p->rstream[0];
    { KLaunch kl(p, "ratio_rhs"); ratio_rhs_kernel<<<dim3((n + 255) / 256, m), 256, 0, st>>>(E, n, LL); }
    if (par) cudaEventRecord(p->ev_rfork, st);
    for (int k = 0; k < m; k++) {
        cudaStream_t sk = (par && k > 0) ? p->rstream[k - 1] : st;
        if (par && k > 0) cudaStreamWaitEvent(sk, p->ev_rfork, 0);
        cudaError_t e = launch_trisolve(p, E + (size_t)k * n, Z + (size_t)k * n, sk, (par && k > 0) ? W + (size_t)(k - 1) * 2 * wsz : nullptr);
        if (e != cudaSuccess) return e;
        if (par && k > 0) { cudaEventRecord(p->ev_rjoin[k - 1], sk); cudaStreamWaitEvent(st, p->ev_rjoin[k - 1], 0); }
    }
    return cudaGetLastError();
}

// c holds the free solution on entry and the constrained one on return
cudaError_t launch_ratio_apply(sfft_plan *p, const double *Z, double *c, cudaStream_t st) {
    const int n = p->g.n, LL = p->g.L * p->g.L, m = p->g.NK - 1;
    if (m < 1) return cudaSuccess;
    KLaunch kl(p, "ratio_apply");
    ratio_apply_kernel<<<1, 256, 0, st>>>(Z, c, n, LL, m);
    return cudaGetLastError();
}

} // namespace sfft
