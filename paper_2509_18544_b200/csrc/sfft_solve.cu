// sfft_solve.cu -- step a4 (BASELINE.json north_star (c), reading C9):
// FP64 solve of G c = h.  G~ = D^-1/2 G D^-1/2 (D = diag G) is factored G~ = L L^T by a
// right-looking blocked Cholesky (block 64): diagonal block in one CTA, panel by triangular
// solve, trailing update C -= X X^T on the FP64 tensor pipe (mma.sync m8n8k4 f64 -- the one
// dense contraction of the path).  A pivot L_kk^2 <= 1e-12 raises the device flag
// (SFFT_ERR_NOT_SPD).  c = D^-1/2 L^-T L^-1 D^-1/2 h by two blocked triangular solves.
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

// diagonal block k0..k0+bs: unblocked right-looking Cholesky in shared memory
__global__ void __launch_bounds__(256) potrf_kernel(double *__restrict__ Lf, int n, int k0, int bs, int *flag) {
    __shared__ double a[CB][CB + 1];
    for (int e = threadIdx.x; e < bs * bs; e += blockDim.x) {
        const int r = e / bs, c = e % bs;
        a[r][c] = Lf[(size_t)(k0 + r) * n + k0 + c];
    }
    for (int j = 0; j < bs; j++) {
        __syncthreads();
        if (threadIdx.x == 0) {
            double s = a[j][j];
            if (!(s > PIVOT_MIN)) { *flag = 1; s = 1.0; }
            a[j][j] = sqrt(s);
        }
        __syncthreads();
        const double d = 1.0 / a[j][j];
        for (int r = j + 1 + threadIdx.x; r < bs; r += blockDim.x) a[r][j] *= d;
        __syncthreads();
        const int m = bs - j - 1;
        for (int e = threadIdx.x; e < m * m; e += blockDim.x) {
            const int r = j + 1 + e / m, c = j + 1 + e % m;
            if (c <= r) a[r][c] -= a[r][j] * a[c][j];
        }
    }
    __syncthreads();
    for (int e = threadIdx.x; e < bs * bs; e += blockDim.x) {
        const int r = e / bs, c = e % bs;
        if (c <= r) Lf[(size_t)(k0 + r) * n + k0 + c] = a[r][c];
    }
}

// panel: rows below the diagonal block, X L_kk^T = A.  grid = ceil(rows/64), block 64 (one row each)
__global__ void __launch_bounds__(CB) trsm_kernel(double *__restrict__ Lf, int n, int k0, int bs) {
    extern __shared__ __align__(16) double dsm[];
    double (*l)[CB + 1] = reinterpret_cast<double (*)[CB + 1]>(dsm);
    double (*x)[CB + 1] = reinterpret_cast<double (*)[CB + 1]>(dsm + CB * (CB + 1));
    const int r0 = k0 + bs + blockIdx.x * CB;
    for (int e = threadIdx.x; e < bs * bs; e += blockDim.x) l[e / bs][e % bs] = Lf[(size_t)(k0 + e / bs) * n + k0 + e % bs];
    for (int e = threadIdx.x; e < CB * bs; e += blockDim.x) {
        const int r = e / bs, c = e % bs;
        x[r][c] = (r0 + r < n) ? Lf[(size_t)(r0 + r) * n + k0 + c] : 0.0;
    }
    __syncthreads();
    const int r = threadIdx.x;
    for (int j = 0; j < bs; j++) {
        double s = x[r][j];
        for (int m = 0; m < j; m++) s = fma(-x[r][m], l[j][m], s);
        x[r][j] = s / l[j][j];
    }
    __syncthreads();
    for (int e = threadIdx.x; e < CB * bs; e += blockDim.x) {
        const int rr = e / bs, c = e % bs;
        if (r0 + rr < n) Lf[(size_t)(r0 + rr) * n + k0 + c] = x[rr][c];
    }
}

__device__ __forceinline__ void dmma884(double &d0, double &d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

// trailing update: for block rows bi >= bj > kb:  A[bi][bj] -= X_bi X_bj^T,  X = panel columns k0..k0+bs.
// grid = ntile*(ntile+1)/2 lower-triangular tile pairs; block 256 = 8 warps, warp tile 16 x 32.
__global__ void __launch_bounds__(256) syrk_kernel(double *__restrict__ Lf, int n, int k0, int bs, int t0 /*first trailing row*/) {
    extern __shared__ __align__(16) double dsm[];
    double (*As)[CLD] = reinterpret_cast<double (*)[CLD]>(dsm);
    double (*Bs)[CLD] = reinterpret_cast<double (*)[CLD]>(dsm + CB * CLD);
    // linear index -> (bi, bj), bj <= bi
    int idx = blockIdx.x, bi = 0;
    while (idx > bi) { idx -= bi + 1; bi++; }
    const int bj = idx;
    const int i0 = t0 + bi * CB, j0 = t0 + bj * CB;
    for (int e = threadIdx.x; e < CB * CB; e += blockDim.x) {
        const int r = e / CB, c = e % CB;
        As[r][c] = (i0 + r < n && c < bs) ? Lf[(size_t)(i0 + r) * n + k0 + c] : 0.0;
        Bs[r][c] = (j0 + r < n && c < bs) ? Lf[(size_t)(j0 + r) * n + k0 + c] : 0.0;
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
#pragma unroll
    for (int a = 0; a < 2; a++)
#pragma unroll
        for (int b = 0; b < 4; b++) {
            const int r = i0 + rw + 8 * a + fr, c = j0 + cw + 8 * b + 2 * fk;
            if (r < n) {
                if (c < n && c <= r) Lf[(size_t)r * n + c] -= acc[a][b][0];
                if (c + 1 < n && c + 1 <= r) Lf[(size_t)r * n + c + 1] -= acc[a][b][1];
            }
        }
}

// ---- triangular solves, single CTA of 1024 threads (32 warps), block 64 ---------------------------
// forward (left-looking): y_blk = L_kk^-1 ( (D h)_blk - L[blk, 0:k0] y[0:k0] )
// backward:               z_blk = L_kk^-T ( y_blk - L[k0+bs:, blk]^T z[k0+bs:] ),  c = D z
__global__ void __launch_bounds__(1024) trisolve_kernel(const double *__restrict__ Lf, const double *__restrict__ dscale,
                                                       const double *__restrict__ h, double *__restrict__ y,
                                                       double *__restrict__ c, int n) {
    __shared__ double blk[CB];
    __shared__ double part[16][CB];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = blockDim.x >> 5;
    const int nblk = (n + CB - 1) / CB;
    // ---------------- forward
    for (int kb = 0; kb < nblk; kb++) {
        const int k0 = kb * CB, bs = min(CB, n - k0);
        for (int r = warp; r < bs; r += nw) {
            const double *row = Lf + (size_t)(k0 + r) * n;
            double s = 0.0;
            for (int j = lane; j < k0; j += 32) s = fma(row[j], y[j], s);
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) s += __shfl_down_sync(0xffffffffu, s, off);
            if (lane == 0) blk[r] = dscale[k0 + r] * h[k0 + r] - s;
        }
        __syncthreads();
        if (warp == 0) {
            // sequential substitution inside the block, lanes over the rows being updated
            for (int j = 0; j < bs; j++) {
                const double xj = blk[j] / Lf[(size_t)(k0 + j) * n + k0 + j];
                __syncwarp();
                if (lane == 0) blk[j] = xj;
                for (int r = j + 1 + lane; r < bs; r += 32) blk[r] -= Lf[(size_t)(k0 + r) * n + k0 + j] * xj;
                __syncwarp();
            }
        }
        __syncthreads();
        for (int r = threadIdx.x; r < bs; r += blockDim.x) y[k0 + r] = blk[r];
        __syncthreads();
    }
    // ---------------- backward
    for (int kb = nblk - 1; kb >= 0; kb--) {
        const int k0 = kb * CB, bs = min(CB, n - k0), t0 = k0 + bs;
        // s[col] = sum_{i >= t0} L[i][k0+col] z[i]: thread -> (col = tid % 64, slice = tid / 64)
        {
            const int col = threadIdx.x & (CB - 1), slice = threadIdx.x >> 6; // 16 slices
            double s = 0.0;
            if (col < bs)
                for (int i = t0 + slice; i < n; i += 16) s = fma(Lf[(size_t)i * n + k0 + col], c[i], s);
            part[slice][col] = s;
        }
        __syncthreads();
        if (threadIdx.x < bs) {
            double s = 0.0;
#pragma unroll
            for (int k = 0; k < 16; k++) s += part[k][threadIdx.x];
            blk[threadIdx.x] = y[k0 + threadIdx.x] - s;
        }
        __syncthreads();
        if (warp == 0) {
            for (int j = bs - 1; j >= 0; j--) {
                const double xj = blk[j] / Lf[(size_t)(k0 + j) * n + k0 + j];
                __syncwarp();
                if (lane == 0) blk[j] = xj;
                for (int r = lane; r < j; r += 32) blk[r] -= Lf[(size_t)(k0 + j) * n + k0 + r] * xj;
                __syncwarp();
            }
        }
        __syncthreads();
        for (int r = threadIdx.x; r < bs; r += blockDim.x) c[k0 + r] = blk[r]; // z, unscaled, read by later blocks
        __syncthreads();
    }
    for (int r = threadIdx.x; r < n; r += blockDim.x) c[r] *= dscale[r];
}

cudaError_t launch_factor(sfft_plan *p) {
    const int n = p->g.n;
    cudaStream_t st = p->stream;
    cudaMemsetAsync(p->flag, 0, sizeof(int), st);
    { KLaunch kl(p, "equil_diag"); equil_diag_kernel<<<(n + 255) / 256, 256, 0, st>>>(p->G, p->dscale, n, p->flag); }
    const long long total = (long long)n * n;
    { KLaunch kl(p, "equil_scale"); equil_scale_kernel<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(p->G, p->dscale, p->Lf, n); }
    const int nblk = (n + CB - 1) / CB;
    const size_t sm_trsm = 2 * CB * (CB + 1) * sizeof(double), sm_syrk = 2 * CB * CLD * sizeof(double);
    cudaFuncSetAttribute(trsm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm_trsm);
    cudaFuncSetAttribute(syrk_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm_syrk);
    for (int kb = 0; kb < nblk; kb++) {
        const int k0 = kb * CB, bs = n - k0 < CB ? n - k0 : CB;
        { KLaunch kl(p, "potrf"); potrf_kernel<<<1, 256, 0, st>>>(p->Lf, n, k0, bs, p->flag); }
        const int rem = n - k0 - bs;
        if (rem > 0) {
            const int nt = (rem + CB - 1) / CB;
            { KLaunch kl(p, "trsm"); trsm_kernel<<<nt, CB, sm_trsm, st>>>(p->Lf, n, k0, bs); }
            { KLaunch kl(p, "syrk"); syrk_kernel<<<nt * (nt + 1) / 2, 256, sm_syrk, st>>>(p->Lf, n, k0, bs, k0 + bs); }
        }
    }
    cudaMemcpyAsync(p->flag_host, p->flag, sizeof(int), cudaMemcpyDeviceToHost, st);
    return cudaGetLastError();
}

cudaError_t launch_trisolve(sfft_plan *p, const double *h, double *c) {
    { KLaunch kl(p, "trisolve"); trisolve_kernel<<<1, 1024, 0, p->stream>>>(p->Lf, p->dscale, h, p->ywork, c, p->g.n); }
    return cudaGetLastError();
}

} // namespace sfft
