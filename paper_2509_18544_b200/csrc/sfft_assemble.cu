// sfft_assemble.cu -- the polynomial terms of a2 and the gather a3
// (BASELINE.json north_star (b)):
//   Gamma_{t,s}[u,v] = X(T_t, P_s)[u,v],  P_s = xt^p yt^q (never masked, reading C7)
//   Delta_s          = sum P_s (m.S)
//   G[(t,u,v),(t',u',v')] = Omega_{tt'}[u-u', v-v'],  G[(t,u,v),s] = Gamma_{t,s}[u,v],  G[s,s'] = Phi_{ss'}
//   h[(t,u,v)] = Theta_t[u,v],  h[s] = Delta_s
// Gamma is separable: with the row moments mu_m[y] = sum_x xt^m (m.R)(x,y) from the a1 row pass,
//   A_{i,p,u}[y] = sum_x xt^i xt((x+u) mod nx)^p (m.R)(x,y)
//               = sum_k C(p,k) (2u/nx)^(p-k) mu_{i+k}[y]  +  (the |u| wrapped pixels, fixed up directly)
//   Gamma_{(i,j),(p,q)}[u,v] = sum_y yt^j yt((y+v) mod ny)^q A_{i,p,u}[y].
#include "sfft_internal.h"

namespace sfft {

__device__ __forceinline__ double ipw(double b, int e) { double r = 1.0; for (int k = 0; k < e; k++) r *= b; return r; }

// one thread per (y, u, i, p)
__global__ void gamma_rows_kernel(const double *__restrict__ mu, const double *__restrict__ R,
                                  const uint8_t *__restrict__ mask, double *__restrict__ gamA, Geom g) {
    const int L = g.L, w = g.w, ny = g.ny, nx = g.nx;
    const long long total = (long long)(g.DK + 1) * (g.DB + 1) * L * ny;
    const long long id = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= total) return;
    const int y = (int)(id % ny);
    long long r = id / ny;
    const int ui = (int)(r % L); r /= L;
    const int pp = (int)(r % (g.DB + 1));
    const int i = (int)(r / (g.DB + 1));
    const int u = ui - w;
    const double delta = 2.0 * u / (double)nx;
    // binomial expansion of (xt + delta)^p
    double acc = 0.0, binom = 1.0;
    for (int k = 0; k <= pp; k++) {
        acc += binom * ipw(delta, pp - k) * mu[(size_t)(i + k) * ny + y];
        binom = binom * (pp - k) / (k + 1);
    }
    // wrapped pixels: xt((x+u) mod nx) = xt + delta -/+ 2
    if (pp > 0 && u != 0) {
        const int xa = u > 0 ? nx - u : 0, xb = u > 0 ? nx : -u;
        for (int x = xa; x < xb; x++) {
            const size_t o = (size_t)y * nx + x;
            double v = R[o]; if (mask && !mask[o]) v = 0.0;
            const double xt = (2.0 * x + 1.0 - nx) / nx;
            const int xw = u > 0 ? x + u - nx : x + u + nx;
            const double xtw = (2.0 * xw + 1.0 - nx) / nx;
            acc += (ipw(xtw, pp) - ipw(xt + delta, pp)) * ipw(xt, i) * v;
        }
    }
    gamA[id] = acc; // layout [i][p][u][y]
}

__device__ __forceinline__ double block_sum2(double v, double *sh) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v += __shfl_down_sync(0xffffffffu, v, off);
    __syncthreads();
    if (lane == 0) sh[wid] = v;
    __syncthreads();
    double r = 0.0;
    if (threadIdx.x == 0) for (int k = 0; k < (int)(blockDim.x >> 5); k++) r += sh[k];
    return r;
}

// Gamma_{(i,j),(p,q)}[u,v] = sum_y W_{j,q,v}[y] A_{i,p,u}[y],  W = yt^j yt((y+v) mod ny)^q: per (t, s) an L x L x ny product.
// gamma_part: grid = (ceil(ny / GC_Y), NB, NK); block = L^2 rounded up to warps.  A CTA brings its GC_Y-row chunk of the L
// rows A_{i,p,.} into shared memory ONCE, forms the L weight rows there, and thread (v, u) takes one dot product; a second
// kernel adds the chunk partials in a fixed order.  (One CTA per (u, v, s, t) re-read the 3 MB table A 44 times through L2
// and repeated the powers 4356 times: 44 us at L = 11, 167-181 us at L = 21, on the tail behind the Omega pass.)
constexpr int GC_Y = 256;
__global__ void gamma_part_kernel(const double *__restrict__ gamA, double *__restrict__ part, Geom g) {
    extern __shared__ __align__(16) double gsm[];
    const int L = g.L, w = g.w, ny = g.ny, LL = L * L;
    double (*As)[GC_Y + 1] = reinterpret_cast<double (*)[GC_Y + 1]>(gsm);
    double (*Ws)[GC_Y + 1] = reinterpret_cast<double (*)[GC_Y + 1]>(gsm + (size_t)L * (GC_Y + 1));
    const int ch = blockIdx.x, s = blockIdx.y, t = blockIdx.z, y0 = ch * GC_Y;
    const int i = g.pi[t], j = g.pj[t], pp = g.pi[s], qq = g.pj[s];
    const double *A = gamA + (((size_t)i * (g.DB + 1) + pp) * L) * ny; // rows u = 0..L-1, ny apart
    const double inv_ny = 1.0 / (double)ny;
    for (int e = threadIdx.x; e < L * GC_Y; e += blockDim.x) {
        const int r = e / GC_Y, yy = e - r * GC_Y, y = y0 + yy;
        double av = 0.0, wv = 0.0;
        if (y < ny) {
            av = A[(size_t)r * ny + y];
            int y2 = y + (r - w); if (y2 >= ny) y2 -= ny; if (y2 < 0) y2 += ny;
            wv = ipw((2.0 * y + 1.0 - ny) * inv_ny, j) * ipw((2.0 * y2 + 1.0 - ny) * inv_ny, qq);
        }
        As[r][yy] = av; Ws[r][yy] = wv;
    }
    __syncthreads();
    const int o = threadIdx.x;
    if (o >= LL) return;
    const int vi = o / L, u = o - vi * L;
    double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;   // four running sums, added in a fixed order
#pragma unroll 4
    for (int yy = 0; yy < GC_Y; yy += 4) {
        a0 = fma(Ws[vi][yy], As[u][yy], a0);
        a1 = fma(Ws[vi][yy + 1], As[u][yy + 1], a1);
        a2 = fma(Ws[vi][yy + 2], As[u][yy + 2], a2);
        a3 = fma(Ws[vi][yy + 3], As[u][yy + 3], a3);
    }
    part[(((size_t)ch * g.NK + t) * g.NB + s) * LL + o] = (a0 + a1) + (a2 + a3);
}
// gam[t][s][v][u] = sum over the chunks, in order
__global__ void gamma_sum_kernel(const double *__restrict__ part, double *__restrict__ gam, int total, int nch) {
    const int id = blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= total) return;
    double v = 0.0;
    for (int c = 0; c < nch; c++) v += part[(size_t)c * total + id];
    gam[id] = v;
}

// grid = NB; block 128:  Delta_s = sum_y yt^q muS_p[y]
__global__ void __launch_bounds__(128) delta_kernel(const double *__restrict__ muS, double *__restrict__ delta, Geom g) {
    __shared__ double sh[32];
    const int s = blockIdx.x, pp = g.pi[s], qq = g.pj[s], ny = g.ny;
    double acc = 0.0;
    for (int y = threadIdx.x; y < ny; y += blockDim.x)
        acc += ipw((2.0 * y + 1.0 - ny) * (1.0 / (double)ny), qq) * muS[(size_t)pp * ny + y];
    acc = block_sum2(acc, sh);
    if (threadIdx.x == 0) delta[s] = acc;
}

__device__ __forceinline__ int pair_index(int t, int tp, int NK) { return t * NK - (t * (t - 1)) / 2 + (tp - t); }

// index meta data of an unknown r < NK L^2: t | (v + w) << 8 | (u + w) << 16; r >= NK L^2 (background term s): -1 - s.
// Geometry only: written once at plan creation (assemble_init), so that the gather of G divides nothing.
__global__ void gather_meta_kernel(int *meta, Geom g) {
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= g.n) return;
    const int L = g.L, LL = L * L, NKLL = g.NK * LL;
    meta[r] = r < NKLL ? ((r / LL) | (((r % LL) / L) << 8) | (((r % LL) % L) << 16)) : -1 - (r - NKLL);
}

// entry (r, c) of G from the lag tables; mr, mc: the meta words of r and c
__device__ __forceinline__ double g_entry(const double *__restrict__ lagO, const double *__restrict__ gam,
                                          const double *__restrict__ phi, const Geom &g, int mr, int mc) {
    const int L = g.L, w = g.w, LL = L * L, W2 = 4 * w + 1;
    if (mr >= 0 && mc >= 0) {
        const int t = mr & 255, v = (mr >> 8) & 255, u = mr >> 16;
        const int tp = mc & 255, vp = (mc >> 8) & 255, up = mc >> 16;
        // X(b,a)[d] = X(a,b)[-d] (pin P11): every entry and its transpose read the SAME table slot, so G is
        // symmetric bit for bit (for t == t' the slot with the lexicographically non-negative lag is used)
        int dv = v - vp, du = u - up;
        const bool flip = t > tp || (t == tp && (dv < 0 || (dv == 0 && du < 0)));
        if (flip) { dv = -dv; du = -du; }
        return lagO[(size_t)pair_index(flip ? tp : t, flip ? t : tp, g.NK) * W2 * W2 + (dv + 2 * w) * W2 + (du + 2 * w)];
    }
    if (mr >= 0) { const int t = mr & 255, v = (mr >> 8) & 255, u = mr >> 16; return gam[((size_t)t * g.NB + (-1 - mc)) * LL + v * L + u]; }
    if (mc >= 0) { const int t = mc & 255, v = (mc >> 8) & 255, u = mc >> 16; return gam[((size_t)t * g.NB + (-1 - mr)) * LL + v * L + u]; }
    return phi[(-1 - mr) * g.NB + (-1 - mc)];
}

// grid = (ceil(n / 256), n): one CTA row per row of G, one thread per entry (both triangles).  The Jacobi equilibration
// of step a4 rides along (the factorisation follows every gather, and two more small launches sat on the critical path
// of a step): the thread also gathers its two diagonal entries and writes the scaled lower triangle
// Lf = D^-1/2 G D^-1/2 and D^-1/2 itself, with the same expressions as equil_diag_kernel / equil_scale_kernel
// (sfft_solve.cu), which remain for a G that arrives some other way.  *flag is raised for a diagonal entry <= 0.
// (With one thread per linear index and its divisions this kernel took 235 us at n = 4416.)
__global__ void __launch_bounds__(256) gather_G_kernel(const double *__restrict__ lagO, const double *__restrict__ gam,
                                const double *__restrict__ phi, const int *__restrict__ meta, double *__restrict__ G,
                                double *__restrict__ Lf, double *__restrict__ dscale, int *flag, Geom g) {
    const int n = g.n, r = blockIdx.y, c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= n) return;
    const int mr = meta[r], mc = meta[c];
    const size_t id = (size_t)r * n + c;
    const double val = g_entry(lagO, gam, phi, g, mr, mc);
    G[id] = val;
    const double grr = g_entry(lagO, gam, phi, g, mr, mr), gcc = g_entry(lagO, gam, phi, g, mc, mc);
    const double sr = grr > 0.0 ? 1.0 / sqrt(grr) : 1.0, sc = gcc > 0.0 ? 1.0 / sqrt(gcc) : 1.0;
    if (c == 0) { dscale[r] = sr; if (!(grr > 0.0)) *flag = 1; }
    Lf[id] = c <= r ? sr * val * sc : 0.0;
}

__global__ void gather_h_kernel(const double *__restrict__ lagT, const double *__restrict__ delta, double *__restrict__ h, Geom g) {
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= g.n) return;
    const int NKLL = g.NK * g.L * g.L;
    h[r] = r < NKLL ? lagT[r] : delta[r - NKLL];
}

cudaError_t launch_gamma(sfft_plan *p) {
    const Geom &g = p->g;
    const long long total = (long long)(g.DK + 1) * (g.DB + 1) * g.L * g.ny;
    { KLaunch kl(p, "gamma_rows"); gamma_rows_kernel<<<(unsigned)((total + 255) / 256), 256, 0, p->cur>>>(p->muR, p->R, p->mask, p->gamA, g); }
    {
        const int nch = (g.ny + GC_Y - 1) / GC_Y, total = g.NK * g.NB * g.L * g.L, bt = ((g.L * g.L + 31) / 32) * 32;
        const size_t sm = (size_t)2 * g.L * (GC_Y + 1) * sizeof(double);
        { KLaunch kl(p, "gamma_cols"); gamma_part_kernel<<<dim3(nch, g.NB, g.NK), bt, sm, p->cur>>>(p->gamA, p->gamP, g); }
        { KLaunch kl(p, "gamma_sum"); gamma_sum_kernel<<<(total + 255) / 256, 256, 0, p->cur>>>(p->gamP, p->gam, total, nch); }
    }
    return cudaGetLastError();
}

cudaError_t launch_delta(sfft_plan *p, const double *muS, double *delta) {
    { KLaunch kl(p, "delta"); delta_kernel<<<p->g.NB, 128, 0, p->cur>>>(muS ? muS : p->muS, delta ? delta : p->delta, p->g); }
    return cudaGetLastError();
}

// plan creation: the index meta data of the gather (p->gmeta allocated by the caller), kernel attributes
cudaError_t assemble_init(sfft_plan *p) {
    {   // gamma_part_kernel: 2 L (GC_Y + 1) doubles of shared memory (86 KB at L = 21)
        const cudaError_t e = cudaFuncSetAttribute(gamma_part_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)((size_t)2 * MAX_L * (GC_Y + 1) * sizeof(double)));
        if (e != cudaSuccess) return e;
    }
    gather_meta_kernel<<<(p->g.n + 255) / 256, 256>>>(p->gmeta, p->g);
    return cudaGetLastError();
}

cudaError_t launch_gather_G(sfft_plan *p) {
    cudaMemsetAsync(p->flag, 0, sizeof(int), p->cur);   // the pivot flag of the factorisation that follows (launch_factor)
    { KLaunch kl(p, "gather_G"); gather_G_kernel<<<dim3((p->g.n + 255) / 256, p->g.n), 256, 0, p->cur>>>(p->lagO, p->gam, p->phi, p->gmeta, p->G, p->Lf, p->dscale, p->flag, p->g); }
    p->lf_ready = true;                                  // Lf and dscale hold the equilibrated matrix of this G
    return cudaGetLastError();
}

cudaError_t launch_gather_h(sfft_plan *p, const double *lagT, const double *delta, double *h) {
    { KLaunch kl(p, "gather_h"); gather_h_kernel<<<(p->g.n + 255) / 256, 256, 0, p->cur>>>(lagT ? lagT : p->lagT, delta ? delta : p->delta, h ? h : p->h, p->g); }
    return cudaGetLastError();
}

} // namespace sfft
