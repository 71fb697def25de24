// sfft_fwd.cu -- step a1 (BASELINE.json north_star (a)):
// polynomial-weighted images xt^i yt^j (m.R) and their 2-D FFTs, plus the FFT of m.S.
//
// T^_(i,j) = FFT_y( yt^j * FFT_x( xt^i * m.R ) ): DK+1 row transforms feed NK column transforms.
// The frame is zero-padded to Mx x My (powers of two); a row of Mx reals is transformed as
// Hx = Mx/2 complex numbers (even/odd packing) and untangled to the half spectrum
// kx = 0..Hx, stored as Hx complex columns with column 0 = X[0] + i X[Hx] (both real).
// The column pass transforms that packed column like any other (it is then the sum
// F0 + i FH of two Hermitian column spectra; consumers untangle it, see sfft_assemble.cu).
#include <cstdlib>
#include "sfft_internal.h"

namespace sfft {

__device__ __forceinline__ double ipow_small(double b, int e) {
    double r = 1.0;
    for (int k = 0; k < e; k++) r *= b;
    return r;
}

// ------------------------------------------------------------------ row pass
// grid.x = ceil(ny / RPB); block = RPB * T threads, T = Hx/E (E values per thread).
// dynamic smem: RPB * padded_lenE<E>(Hx) cplx  +  RPB * 8 * 8 doubles (moment partials)
template <int E, int LOG2N_CT = 0>
__global__ void __launch_bounds__(256, E == 16 ? 2 : 4) row_fwd_kernel(const double *__restrict__ img, const uint8_t *__restrict__ mask,
                                                     cplx *__restrict__ inter, int NI, double *__restrict__ mu, int NMOM,
                                                     Geom g, const cplx *__restrict__ tw) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int Hx = LOG2N_CT ? (1 << LOG2N_CT) : g.Hx, T = Hx / E;
    const int RPB = LOG2N_CT ? 1 : blockDim.x / T; // the fixed-size instances run one row per CTA
    const int rib = LOG2N_CT ? 0 : threadIdx.x / T, j = threadIdx.x - rib * T;
    const int row = blockIdx.x * RPB + rib;
    const bool live = row < g.ny;
    cplx *s = reinterpret_cast<cplx *>(smem_raw) + (size_t)rib * padded_lenE<E>(Hx);
    double *wpart = reinterpret_cast<double *>(reinterpret_cast<cplx *>(smem_raw) + (size_t)RPB * padded_lenE<E>(Hx));
    const double inv_nx = 1.0 / (double)g.nx;
    const size_t rowoff = (size_t)row * g.nx;
    const bool vec = ((g.nx & 1) == 0) && (((size_t)img & 15) == 0);

    for (int i = 0; i < NI; i++) {
        cplx v[E];
        double mom[8];
#pragma unroll
        for (int m = 0; m < 8; m++) mom[m] = 0.0;
#pragma unroll
        for (int q = 0; q < E; q++) {
            const int x0 = 2 * (j + q * T);
            double a = 0.0, b = 0.0;
            if (live) {
                if (vec) { // even nx, 16-byte aligned image: one 16-byte load per pixel pair
                    if (x0 < g.nx) { const double2 ab = *reinterpret_cast<const double2 *>(img + rowoff + x0); a = ab.x; b = ab.y; }
                } else {
                    if (x0 < g.nx) a = img[rowoff + x0];
                    if (x0 + 1 < g.nx) b = img[rowoff + x0 + 1];
                }
                if (mask) {
                    if (x0 < g.nx && !mask[rowoff + x0]) a = 0.0;
                    if (x0 + 1 < g.nx && !mask[rowoff + x0 + 1]) b = 0.0;
                }
            }
            const double xa = (2.0 * x0 + 1.0 - g.nx) * inv_nx, xb = (2.0 * x0 + 3.0 - g.nx) * inv_nx;
            if (i == 0 && NMOM > 0) {
                double pa = a, pb = b;
#pragma unroll
                for (int m = 0; m < 8; m++)
                    if (m < NMOM) { mom[m] += pa + pb; pa *= xa; pb *= xb; }
            }
            v[q] = mk(a * ipow_small(xa, i), b * ipow_small(xb, i));
        }
        if (i == 0 && NMOM > 0) {
            // deterministic reduction over the T threads of this row
            const int width = T < 32 ? T : 32;
#pragma unroll
            for (int m = 0; m < 8; m++)
                if (m < NMOM)
                    for (int off = width >> 1; off > 0; off >>= 1) mom[m] += __shfl_down_sync(0xffffffffu, mom[m], off, width);
            const int nw = T > 32 ? (T >> 5) : 1; // warps per row
            if ((j & (width - 1)) == 0) {
                const int wi = T > 32 ? (j >> 5) : 0;
#pragma unroll
                for (int m = 0; m < 8; m++) // static indices: a run-time bound here would push mom[] into local memory
                    if (m < NMOM) wpart[(rib * 8 + wi) * 8 + m] = mom[m];
            }
            __syncthreads();
            if (j == 0 && live)
                for (int m = 0; m < NMOM; m++) {
                    double acc = 0.0;
                    for (int k = 0; k < nw; k++) acc += wpart[(rib * 8 + k) * 8 + m];
                    mu[(size_t)m * g.ny + row] = acc;
                }
        }
        fft_blockE<-1, E, LOG2N_CT>(v, s, g.log2Hx, j, tw, g.Nt);
        __syncthreads();
#pragma unroll
        for (int q = 0; q < E; q++) s[padE<E>(j + q * T)] = v[q];
        __syncthreads();
        // untangle: X[k] = E[k] + exp(-2 pi i k/Mx) O[k],  E = (Z[k] + conj Z[Hx-k])/2, O = (Z[k] - conj Z[Hx-k])/(2i)
        cplx *dst = inter + ((size_t)i * g.ny + row) * Hx;
#pragma unroll
        for (int q = 0; q < E; q++) {
            const int k = j + q * T;
            const cplx A = s[padE<E>(k)], B = cconj(s[padE<E>((Hx - k) & (Hx - 1))]);
            const cplx E = mk(0.5 * (A.x + B.x), 0.5 * (A.y + B.y));
            const cplx O = mk(0.5 * (A.y - B.y), -0.5 * (A.x - B.x));
            cplx X;
            if (k == 0) X = mk(E.x + O.x, E.x - O.x);
            else X = cadd(E, cmul(tw[(size_t)k * (g.Nt / g.Mx)], O));
            if (live) dst[k] = X;
        }
    }
}

// ------------------------------------------------------------------ column pass
// block b -> (spectrum k = b % ns, column group b / ns); C columns per CTA, T = My/16 threads each,
// thread tid -> (c = tid % C, j = tid / C).  dynamic smem: C * padded_len(My) cplx.

__global__ void __launch_bounds__(512) col_fwd_kernel(const cplx *__restrict__ inter, cplx *__restrict__ spec, ColJobs jobs,
                                                     int C, Geom g, const cplx *__restrict__ tw) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int My = g.My, T = My >> 4, Hx = g.Hx;
    const int k = blockIdx.x % jobs.ns, cg = blockIdx.x / jobs.ns;
    const int c = threadIdx.x % C, j = threadIdx.x / C;
    const int col = cg * C + c;
    cplx *s = reinterpret_cast<cplx *>(smem_raw) + (size_t)c * padded_len(My);
    const cplx *src = inter + (size_t)jobs.ii[k] * g.ny * Hx + col;
    const int jp = jobs.jj[k];
    const double inv_ny = 1.0 / (double)g.ny;
    cplx v[16];
#pragma unroll
    for (int q = 0; q < 16; q++) {
        const int row = j + q * T;
        cplx a = mk(0.0, 0.0);
        if (row < g.ny) {
            a = src[(size_t)row * Hx];
            if (jp > 0) a = cscale(a, ipow_small((2.0 * row + 1.0 - g.ny) * inv_ny, jp));
        }
        v[q] = a;
    }
    fft_block<-1>(v, s, g.log2My, j, tw, g.Nt);
    cplx *dst = spec + (size_t)k * My * Hx;
#pragma unroll
    for (int q = 0; q < 16; q++) dst[spec_idx(j + q * T, col, My)] = v[q];
}

// values per thread of the row / column transforms: 8 keeps a thread under 64 registers (twice the
// resident warps of 16) at the price of one more shared-memory exchange; SFFT_ROW_E / SFFT_COL_E override
int fft_E(const char *env, int N, int dflt) {
    int E = dflt;
    if (const char *s = getenv(env)) E = atoi(s) == 8 ? 8 : 16;
    if (N / 8 > 256 && E == 8) E = 16;   // a transform is at most 256 threads
    if (N < 32) E = 8;
    return E;
}

int row_cfg(const Geom &g, int E, int *threads, size_t *smem) {
    const int T = g.Hx / E;
    int RPB = 64 / T; if (RPB < 1) RPB = 1;   // one row per CTA once a row has >= 64 threads: several small CTAs per SM
    *threads = RPB * T;                        // run in different phases (load / butterflies / store) and overlap
    *smem = (size_t)RPB * (E == 8 ? padded_lenE<8>(g.Hx) : padded_lenE<16>(g.Hx)) * sizeof(cplx) + (size_t)RPB * 64 * sizeof(double);
    return RPB;
}

int col_cfg(const Geom &g, int *threads, size_t *smem) {
    const int T = g.My >> 4;
    int C = 512 / T; if (C < 1) C = 1; if (C > g.Hx) C = g.Hx;
    *threads = C * T;
    *smem = (size_t)C * padded_len(g.My) * sizeof(cplx);
    return C;
}

cudaError_t launch_row_fwd(sfft_plan *p, const double *img, const uint8_t *mask, cplx *inter, int NI, double *mu, int NMOM) {
    const Geom &g = p->g;
    int threads; size_t smem;
    const int E = fft_E("SFFT_ROW_E", g.Hx, 8);
    const int RPB = row_cfg(g, E, &threads, &smem);
    static bool attr_set = false;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(row_fwd_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(row_fwd_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(row_fwd_kernel<8, 11>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    {
        KLaunch kl(p, NI > 1 ? "row_fwd_R" : "row_fwd_S");
        if (E == 8 && g.log2Hx == 11 && RPB == 1) row_fwd_kernel<8, 11><<<g.ny, threads, smem, p->stream>>>(img, mask, inter, NI, mu, NMOM, g, p->tw);
        else if (E == 8) row_fwd_kernel<8><<<(g.ny + RPB - 1) / RPB, threads, smem, p->stream>>>(img, mask, inter, NI, mu, NMOM, g, p->tw);
        else row_fwd_kernel<16><<<(g.ny + RPB - 1) / RPB, threads, smem, p->stream>>>(img, mask, inter, NI, mu, NMOM, g, p->tw);
    }
    return cudaGetLastError();
}

cudaError_t launch_col_fwd(sfft_plan *p, const cplx *inter, cplx *spec, int ns, const int *ii, const int *jj) {
    const Geom &g = p->g;
    if (colpipe_ok(g)) {
        int nsrc = 0;
        for (int k = 0; k < ns; k++) if (ii[k] + 1 > nsrc) nsrc = ii[k] + 1;
        return launch_colpipe_fwd(p, inter, spec, ns, ii, jj, nsrc);
    }
    int threads; size_t smem;
    const int C = col_cfg(g, &threads, &smem);
    static bool attr_set = false;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(col_fwd_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    ColJobs jobs; jobs.ns = ns;
    for (int k = 0; k < ns; k++) { jobs.ii[k] = ii[k]; jobs.jj[k] = jj[k]; }
    { KLaunch kl(p, ns > 1 ? "col_fwd_R" : "col_fwd_S"); col_fwd_kernel<<<ns * (g.Hx / C), threads, smem, p->stream>>>(inter, spec, jobs, C, g, p->tw); }
    return cudaGetLastError();
}

} // namespace sfft
