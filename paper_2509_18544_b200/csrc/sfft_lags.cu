// sfft_lags.cu -- step a2 (BASELINE.json north_star (b)):
// cross-correlations X(a,b)[du,dv] = sum_{x,y} a(x,y) b((x+du) mod nx, (y+dv) mod ny) of the
// polynomial-weighted images, read off at the kernel-offset pairs only, from the spectra.
//
//   X_M(a,b)[du,dv] = 1/(Mx My) sum_{ky} sum_{kx=0..Hx} g(kx) Re( conj(A) B e^{2 pi i (kx du/Mx + ky dv/My)} )
//
// (g = 1 for kx = 0, Hx, else 2: Hermitian symmetry of real images) is the Mx x My-circular
// correlation of the ZERO-PADDED images.  It is turned into the nx x ny-circular correlation
// the method defines (reading C6) by adding the few products that wrap differently:
//   X_N - X_M = sum over pixels with x+du or y+dv outside the frame of
//               a(x,y) * ( b((x+du) mod nx, (y+dv) mod ny) - bpad((x+du) mod Mx, (y+dv) mod My) ).
// The product spectrum and the correlation image are never materialised: the inverse
// transform is pruned to the (2W+1)^2 lags that are used (output-pruned DFT).
//
// Kernels:
//   lagcol_kernel  stage 1: Q[p][dv][kx] = sum_ky conj(A)B e^{2 pi i ky dv/My}, thread = (pair, kx),
//                  rows streamed through a cp.async shared-memory pipeline shared by all pairs
//   lagedge_kernel the packed column kx = 0 (DC + i Nyquist) untangled -> Q[.][.][0], Q[.][.][Hx]
//   (sfft_border.cu) the wrap corrections X_N - X_M from border strips
//   lagrow_kernel  stage 2: lag[p][dv][du] = 1/(Mx My) sum_kx g Re(Q e^{2 pi i kx du/Mx}) + border
#include "sfft_internal.h"

namespace sfft {

struct SpecSet { const cplx *p[MAX_NP + 1]; };

__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gsrc) {
    unsigned sa = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(sa), "l"(gsrc));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

constexpr int LC_RT = 8;   // rows per pipeline stage
constexpr int LC_NST = 3;  // stages

// grid = (kx blocks, pair groups, ky splits); block = npg * KXC threads (npg = pairs per group).
// dynamic smem: LC_NST * LC_RT * (ns*KXC + WB) cplx
template <int WB>
__global__ void __launch_bounds__(WB > 10 ? 288 : 512)
lagcol_kernel(SpecSet ss, int ns, PairList pl, int npg, int KXC, int W, int rows_per_split, cplx *__restrict__ Q,
              Geom g, const cplx *__restrict__ tw) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx *tile = reinterpret_cast<cplx *>(smem_raw);
    const int Hx = g.Hx, My = g.My;
    const int stage_elems = LC_RT * (ns * KXC + WB);
    const int kx0 = blockIdx.x * KXC;
    const int pl0 = blockIdx.y * npg;
    const int r0 = blockIdx.z * rows_per_split;
    const int r1 = min(My, r0 + rows_per_split);
    const int nIt = (r1 - r0 + LC_RT - 1) / LC_RT;
    const int lp = threadIdx.x / KXC, lane = threadIdx.x - lp * KXC;
    const int p = pl0 + lp;
    const bool active = (p < pl.np) && (lp < npg);
    const int sa = active ? pl.a[p] : 0, sb = active ? pl.b[p] : 0;
    const int twsy = g.Nt / My;

    double a0r = 0.0, a0i = 0.0;
    double s1[WB], s2[WB], s3[WB], s4[WB];
#pragma unroll
    for (int d = 0; d < WB; d++) { s1[d] = 0.0; s2[d] = 0.0; s3[d] = 0.0; s4[d] = 0.0; }

    auto issue = [&](int it) {
        if (it < nIt) {
            cplx *st = tile + (size_t)(it % LC_NST) * stage_elems;
            const int per_row = ns * KXC + WB;
            for (int e = threadIdx.x; e < stage_elems; e += blockDim.x) {
                const int r = e / per_row, o = e - r * per_row;
                int ky = r0 + it * LC_RT + r; if (ky >= r1) ky = r1 - 1;
                const cplx *src;
                if (o < ns * KXC) {
                    const int s = o / KXC; int kx = kx0 + (o - s * KXC); if (kx >= Hx) kx = Hx - 1;
                    src = ss.p[s] + (size_t)ky * Hx + kx;
                } else {
                    const int d = o - ns * KXC + 1;
                    src = tw + (size_t)((ky * d) & (My - 1)) * twsy;
                }
                cp_async16(st + e, src);
            }
        }
        cp_async_commit();
    };

    for (int it = 0; it < LC_NST - 1; it++) issue(it);
    for (int it = 0; it < nIt; it++) {
        issue(it + LC_NST - 1);
        cp_async_wait<LC_NST - 1>();
        __syncthreads();
        if (active) {
            const cplx *st = tile + (size_t)(it % LC_NST) * stage_elems;
            const int nr = min(LC_RT, r1 - r0 - it * LC_RT);
            for (int r = 0; r < nr; r++) {
                const cplx *row = st + r * (ns * KXC + WB);
                const cplx A = row[sa * KXC + lane], B = row[sb * KXC + lane];
                const double pr = A.x * B.x + A.y * B.y, pi = A.x * B.y - A.y * B.x;
                a0r += pr; a0i += pi;
                const cplx *ph = row + ns * KXC;
#pragma unroll
                for (int d = 0; d < WB; d++) {
                    const cplx e = ph[d];            // exp(-i phi): cos = e.x, sin = -e.y
                    s1[d] = fma(pr, e.x, s1[d]); s2[d] = fma(pi, e.y, s2[d]);
                    s3[d] = fma(pr, e.y, s3[d]); s4[d] = fma(pi, e.x, s4[d]);
                }
            }
        }
        __syncthreads();
    }
    // Q[+d] = (S1 - S2) + i(S3 + S4),  Q[-d] = (S1 + S2) + i(S4 - S3)  with sin = -e.y folded in:
    // s2 = -sum pi*sin, s3 = -sum pr*sin
    const int kx = kx0 + lane;
    if (active && kx < Hx) {
        cplx *q = Q + ((size_t)(blockIdx.z * pl.np + p) * (2 * W + 1)) * (Hx + 1) + kx;
        q[(size_t)W * (Hx + 1)] = mk(a0r, a0i);
#pragma unroll
        for (int d = 0; d < WB; d++)
            if (d < W) {
                q[(size_t)(W + d + 1) * (Hx + 1)] = mk(s1[d] + s2[d], s4[d] - s3[d]);
                q[(size_t)(W - d - 1) * (Hx + 1)] = mk(s1[d] - s2[d], s4[d] + s3[d]);
            }
    }
}

// deterministic block sum of one double per thread (blockDim.x <= 1024, power of two)
__device__ __forceinline__ double block_sum(double v, double *sh) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v += __shfl_down_sync(0xffffffffu, v, off);
    __syncthreads();
    if (lane == 0) sh[wid] = v;
    __syncthreads();
    double r = 0.0;
    if (threadIdx.x == 0) for (int k = 0; k < (int)(blockDim.x >> 5); k++) r += sh[k];
    return r; // valid in thread 0
}

// grid = (np, 2W+1); block 256.  Column 0 holds F = F0 + i FH (F0, FH: column spectra of the real
// columns kx = 0 and kx = Hx of the row transform): F0[ky] = (F[ky] + conj F[-ky])/2,
// FH[ky] = (F[ky] - conj F[-ky])/(2i).
__global__ void __launch_bounds__(256) lagedge_kernel(SpecSet ss, PairList pl, int W, int nsplit, cplx *__restrict__ Q,
                                                     Geom g, const cplx *__restrict__ tw) {
    __shared__ double sh[32];
    const int p = blockIdx.x, dv = (int)blockIdx.y - W;
    const int Hx = g.Hx, My = g.My;
    const cplx *FA = ss.p[pl.a[p]], *FB = ss.p[pl.b[p]];
    double q0r = 0, q0i = 0, qhr = 0, qhi = 0;
    for (int ky = threadIdx.x; ky < My; ky += blockDim.x) {
        const int kn = (My - ky) & (My - 1);
        const cplx a = FA[(size_t)ky * Hx], am = cconj(FA[(size_t)kn * Hx]);
        const cplx b = FB[(size_t)ky * Hx], bm = cconj(FB[(size_t)kn * Hx]);
        const cplx A0 = mk(0.5 * (a.x + am.x), 0.5 * (a.y + am.y)), AH = mk(0.5 * (a.y - am.y), -0.5 * (a.x - am.x));
        const cplx B0 = mk(0.5 * (b.x + bm.x), 0.5 * (b.y + bm.y)), BH = mk(0.5 * (b.y - bm.y), -0.5 * (b.x - bm.x));
        cplx e = tw[(size_t)((ky * (dv + My)) & (My - 1)) * (g.Nt / My)];
        e.y = -e.y; // exp(+2 pi i ky dv/My)
        const cplx P0 = cmul(cmulc(A0, B0), e), PH = cmul(cmulc(AH, BH), e);
        q0r += P0.x; q0i += P0.y; qhr += PH.x; qhi += PH.y;
    }
    q0r = block_sum(q0r, sh); q0i = block_sum(q0i, sh); qhr = block_sum(qhr, sh); qhi = block_sum(qhi, sh);
    if (threadIdx.x == 0)
        for (int s = 0; s < nsplit; s++) {
            cplx *q = Q + ((size_t)(s * pl.np + p) * (2 * W + 1) + blockIdx.y) * (Hx + 1);
            q[0] = s == 0 ? mk(q0r, q0i) : mk(0, 0);
            q[Hx] = s == 0 ? mk(qhr, qhi) : mk(0, 0);
        }
}

// ---------------------------------------------------------------- stage 2
// grid = (np, 2W+1 [dv]); block 256.
__global__ void __launch_bounds__(256) lagrow_kernel(const cplx *__restrict__ Q, int np, int W, int nsplit,
                                                    const double *__restrict__ bpart, int nchunk,
                                                    double *__restrict__ lag, Geom g, const cplx *__restrict__ tw) {
    __shared__ double sh[32];
    const int p = blockIdx.x, dvi = blockIdx.y, Hx = g.Hx, Mx = g.Mx;
    constexpr int WM = MAX_L - 1; // 20
    double sc[WM + 1], sn[WM + 1];
#pragma unroll
    for (int d = 0; d <= WM; d++) { sc[d] = 0.0; sn[d] = 0.0; }
    for (int kx = threadIdx.x; kx <= Hx; kx += blockDim.x) {
        cplx q = mk(0, 0);
        for (int s = 0; s < nsplit; s++) q = cadd(q, Q[((size_t)(s * np + p) * (2 * W + 1) + dvi) * (Hx + 1) + kx]);
        const double gw = (kx == 0 || kx == Hx) ? 1.0 : 2.0;
        q.x *= gw; q.y *= gw;
#pragma unroll
        for (int d = 0; d <= WM; d++)
            if (d <= W) {
                const cplx e = tw[(size_t)((kx * d) & (Mx - 1)) * (g.Nt / Mx)]; // cos = e.x, sin = -e.y
                sc[d] = fma(q.x, e.x, sc[d]); sn[d] = fma(q.y, -e.y, sn[d]);
            }
    }
    const double scale = 1.0 / ((double)g.Mx * (double)g.My);
    const int nl = (2 * W + 1) * (2 * W + 1);
    for (int d = 0; d <= W; d++) {
        double c = 0.0, s = 0.0;
#pragma unroll
        for (int k = 0; k <= WM; k++) if (k == d) { c = sc[k]; s = sn[k]; }
        c = block_sum(c, sh); s = block_sum(s, sh);
        if (threadIdx.x == 0) {
            double vp = (c - s) * scale, vm = (c + s) * scale; // Re(q e^{+i th}), Re(q e^{-i th})
            const int ip = dvi * (2 * W + 1) + (W + d), im = dvi * (2 * W + 1) + (W - d);
            for (int k = 0; k < nchunk; k++) {
                vp += bpart[((size_t)k * np + p) * nl + ip];
                if (d > 0) vm += bpart[((size_t)k * np + p) * nl + im];
            }
            lag[(size_t)p * nl + ip] = vp;
            if (d > 0) lag[(size_t)p * nl + im] = vm;
        }
    }
}

// ---------------------------------------------------------------- host side
// Launch shape of stage 1 (also used by the plan to size Q).
void lagcol_config(const Geom &g, int np, int W, LagCfg *c) {
    const int WB = W <= 3 ? 3 : W <= 5 ? 5 : W <= 6 ? 6 : W <= 10 ? 10 : 20;
    const int maxthreads = WB > 10 ? 288 : 512;
    int KXC = maxthreads / np, npg = np;
    if (KXC < 8) { KXC = 8; npg = maxthreads / KXC; }   // split the pairs into groups, keep 128-byte runs
    if (KXC > 32) KXC = 32;
    if (WB <= 10 && np * 14 <= maxthreads && np * 16 > 256 && g.Hx >= 1024) KXC = 14; // Hx=2048: 147 CTAs on 148 SMs
    if (KXC > g.Hx) KXC = g.Hx;
    const int nkb = (g.Hx + KXC - 1) / KXC, ngr = (np + npg - 1) / npg;
    int nsplit = 1;
    while (nkb * ngr * nsplit < 148 && nsplit < 8 && g.My / (nsplit * 2) >= 64) nsplit *= 2;
    c->WB = WB; c->KXC = KXC; c->npg = npg; c->nkb = nkb; c->ngr = ngr; c->nsplit = nsplit;
    c->rows_per_split = (g.My + nsplit - 1) / nsplit;
}

template <int WB>
static cudaError_t run_lagcol(sfft_plan *p, const SpecSet &ss, int ns, const PairList &pl, int W, const LagCfg &c, bool science) {
    const Geom &g = p->g;
    const size_t smem = (size_t)LC_NST * LC_RT * (ns * c.KXC + WB) * sizeof(cplx);
    cudaError_t e = cudaFuncSetAttribute(lagcol_kernel<WB>, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024);
    if (e != cudaSuccess) return e;
    dim3 grid(c.nkb, c.ngr, c.nsplit);
    { KLaunch kl(p, science ? "lagcol_theta" : "lagcol_omega"); lagcol_kernel<WB><<<grid, c.npg * c.KXC, smem, p->stream>>>(ss, ns, pl, c.npg, c.KXC, W, c.rows_per_split, p->Q, g, p->tw); }
    return cudaGetLastError();
}

int border_chunks() { return 1; }

cudaError_t launch_lags(sfft_plan *p, const PairList &pl, int W, double *lag, bool science) {
    const Geom &g = p->g;
    SpecSet ss;
    for (int t = 0; t < g.NK; t++) ss.p[t] = p->specT + (size_t)t * g.My * g.Hx;
    ss.p[g.NK] = p->specS;
    const int ns = science ? g.NK + 1 : g.NK;
    LagCfg c; lagcol_config(g, pl.np, W, &c);
    const int nsplit = c.nsplit;
    cudaError_t e;
    if (c.WB == 3) e = run_lagcol<3>(p, ss, ns, pl, W, c, science);
    else if (c.WB == 5) e = run_lagcol<5>(p, ss, ns, pl, W, c, science);
    else if (c.WB == 6) e = run_lagcol<6>(p, ss, ns, pl, W, c, science);
    else if (c.WB == 10) e = run_lagcol<10>(p, ss, ns, pl, W, c, science);
    else e = run_lagcol<20>(p, ss, ns, pl, W, c, science);
    if (e != cudaSuccess) return e;
    { KLaunch kl(p, science ? "lagedge_theta" : "lagedge_omega"); lagedge_kernel<<<dim3(pl.np, 2 * W + 1), 256, 0, p->stream>>>(ss, pl, W, nsplit, p->Q, g, p->tw); }
    int nchunk = 0;
    double *bpart = p->bpart;
    if (g.Mx != g.nx || g.My != g.ny) {
        nchunk = border_chunks();
        if (W > 0) { e = launch_border(p, pl, W, science, bpart); if (e != cudaSuccess) return e; }
        else nchunk = 0;
    }
    { KLaunch kl(p, science ? "lagrow_theta" : "lagrow_omega"); lagrow_kernel<<<dim3(pl.np, 2 * W + 1), 256, 0, p->stream>>>(p->Q, pl.np, W, nsplit, bpart, nchunk, lag, g, p->tw); }
    return cudaGetLastError();
}

} // namespace sfft
