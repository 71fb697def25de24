// sfft_subtract.cu -- step a5 (BASELINE.json north_star (d)):
//   M = sum_t T_t (*) K_t  (circular at nx x ny, T_t = xt^i yt^j R UNMASKED, K_t[u,v] = a_{t,u,v}),
//   D = S - M - B,  B = sum_s b_s xt^p yt^q.
// By FFT on the zero-padded Mx x My grid:  M^ = sum_t T^_t K^_t,
//   K^_t[ky,kx] = sum_v e^{-2 pi i ky v/My} E_t[v][kx],  E_t[v][kx] = sum_u a_{t,u,v} e^{-2 pi i kx u/Mx}.
// Kernels:
//   ktab_kernel     coefficients -> row tables, stored folded over +-v:
//                   slot 0: E[0];  slot 2v-1: E[v]+E[-v];  slot 2v: -i (E[v]-E[-v])   (v = 1..w)
//                   so that K^ = slot0 + sum_v cos(th v) slot(2v-1) + sin(th v) slot(2v),  th = 2 pi ky/My
//   col_inv_kernel  M^ column by column (K^ synthesised on the fly) + inverse FFT along y
//   row_inv_kernel  Hermitian -> packed, inverse FFT along x, fused D = S - M - B
//   wrapfix_kernel  pixels within w of the frame edge: replace the taps that wrap on the padded
//                   grid by the taps that wrap on the native grid (reading C6)
#include "sfft_internal.h"

namespace sfft {

// grid = (ceil((Hx+1)/128), w+1, NK); block 128
__global__ void __launch_bounds__(128) ktab_kernel(const double *__restrict__ coef, cplx *__restrict__ E, Geom g,
                                                  const cplx *__restrict__ tw) {
    const int kx = blockIdx.x * blockDim.x + threadIdx.x;
    if (kx > g.Hx) return;
    const int v = blockIdx.y, t = blockIdx.z, L = g.L, w = g.w, Mx = g.Mx;
    const double *ap = coef + (size_t)t * L * L + (size_t)(w + v) * L + w; // a_{t,u,+v} at ap[u]
    const double *am = coef + (size_t)t * L * L + (size_t)(w - v) * L + w; // a_{t,u,-v}
    cplx ep = mk(0, 0), em = mk(0, 0);
    for (int u = -w; u <= w; u++) {
        const cplx e = tw[(size_t)((kx * (u + Mx)) & (Mx - 1)) * (g.Nt / Mx)]; // exp(-2 pi i kx u/Mx)
        ep.x = fma(ap[u], e.x, ep.x); ep.y = fma(ap[u], e.y, ep.y);
        em.x = fma(am[u], e.x, em.x); em.y = fma(am[u], e.y, em.y);
    }
    cplx *Et = E + (size_t)t * L * (g.Hx + 1);
    if (v == 0) Et[kx] = ep;
    else {
        Et[(size_t)(2 * v - 1) * (g.Hx + 1) + kx] = cadd(ep, em);
        const cplx d = csub(ep, em);
        Et[(size_t)(2 * v) * (g.Hx + 1) + kx] = mk(d.y, -d.x); // -i d
    }
}

// K^ at (phase powers ph[v-1] = exp(-i th v)) from the folded table column e[slot*estride]
__device__ __forceinline__ cplx khat(const cplx *e, int estride, int w, const double *cs, const double *sn) {
    cplx k = e[0];
    for (int v = 1; v <= w; v++) {
        const cplx p = e[(2 * v - 1) * estride], m = e[(2 * v) * estride];
        k.x = fma(cs[v - 1], p.x, k.x); k.y = fma(cs[v - 1], p.y, k.y);
        k.x = fma(sn[v - 1], m.x, k.x); k.y = fma(sn[v - 1], m.y, k.y);
    }
    return k;
}

constexpr int MAXW = (MAX_L - 1) / 2;

// block b -> column group; C columns per CTA, T = My/16 threads per column, tid -> (c = tid % C, j = tid / C).
// dynamic smem: C*padded_len(My) cplx (FFT)  +  NK*L*(C+1) cplx (folded tables of the CTA's columns; slot C = kx=Hx)
__global__ void __launch_bounds__(512) col_inv_kernel(const cplx *__restrict__ spec, const cplx *__restrict__ E,
                                                     cplx *__restrict__ inter, int C, Geom g, const cplx *__restrict__ tw) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int My = g.My, T = My >> 4, Hx = g.Hx, L = g.L, w = g.w, NK = g.NK;
    const int c = threadIdx.x % C, j = threadIdx.x / C;
    const int col0 = blockIdx.x * C, col = col0 + c;
    cplx *s = reinterpret_cast<cplx *>(smem_raw) + (size_t)c * padded_len(My);
    cplx *et = reinterpret_cast<cplx *>(smem_raw) + (size_t)C * padded_len(My);
    const int es = C + 1;
    for (int e = threadIdx.x; e < NK * L * es; e += blockDim.x) {
        const int cc = e % es, sl = e / es; // sl = t*L + slot
        const int kx = cc < C ? col0 + cc : Hx;
        et[e] = E[(size_t)sl * (Hx + 1) + kx];
    }
    __syncthreads();
    const size_t plane = (size_t)My * Hx;
    const int twsy = g.Nt / My;
    cplx v[16];
#pragma unroll 2
    for (int q = 0; q < 16; q++) {
        const int ky = j + q * T;
        double cs[MAXW], sn[MAXW];
        {
            const cplx p1 = tw[(size_t)ky * twsy]; // exp(-i th): cos = x, sin = -y
            cplx p = p1;
            for (int vv = 0; vv < w; vv++) { cs[vv] = p.x; sn[vv] = -p.y; p = cmul(p, p1); }
        }
        cplx acc = mk(0, 0);
        if (col != 0) {
            for (int t = 0; t < NK; t++) {
                const cplx k = khat(et + (size_t)t * L * es + c, es, w, cs, sn);
                acc = cadd(acc, cmul(spec[(size_t)t * plane + spec_idx(ky, col, My)], k));
            }
        } else {
            // packed column: Z = F0 + i FH  ->  M0 = sum F0 K^(kx=0), MH = sum FH K^(kx=Hx), repacked M0 + i MH
            const int kn = (My - ky) & (My - 1);
            cplx a0 = mk(0, 0), aH = mk(0, 0);
            for (int t = 0; t < NK; t++) {
                const cplx z = spec[(size_t)t * plane + spec_idx(ky, 0, My)], zm = cconj(spec[(size_t)t * plane + spec_idx(kn, 0, My)]);
                const cplx F0 = mk(0.5 * (z.x + zm.x), 0.5 * (z.y + zm.y)), FH = mk(0.5 * (z.y - zm.y), -0.5 * (z.x - zm.x));
                a0 = cadd(a0, cmul(F0, khat(et + (size_t)t * L * es + 0, es, w, cs, sn)));
                aH = cadd(aH, cmul(FH, khat(et + (size_t)t * L * es + C, es, w, cs, sn)));
            }
            acc = mk(a0.x - aH.y, a0.y + aH.x);
        }
        v[q] = acc;
    }
    fft_block<1>(v, s, g.log2My, j, tw, g.Nt);
#pragma unroll
    for (int q = 0; q < 16; q++) {
        const int row = j + q * T;
        if (row < g.ny) inter[(size_t)row * Hx + col] = v[q];
    }
}

// grid.x = ceil(ny/RPB); block = RPB*T, T = Hx/E.  dynamic smem: RPB*padded_lenE<E>(Hx) cplx
template <int E, int LOG2N_CT = 0>
__global__ void __launch_bounds__(256, E == 16 ? 2 : 4) row_inv_kernel(const cplx *__restrict__ inter, const double *__restrict__ S,
                                                     const double *__restrict__ coef, double *__restrict__ D, Geom g,
                                                     const cplx *__restrict__ tw, int mode) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int Hx = LOG2N_CT ? (1 << LOG2N_CT) : g.Hx, T = Hx / E;
    const int RPB = LOG2N_CT ? 1 : blockDim.x / T;
    const int rib = LOG2N_CT ? 0 : threadIdx.x / T, j = threadIdx.x - rib * T;
    const int row = blockIdx.x * RPB + rib;
    const bool live = row < g.ny;
    cplx *s = reinterpret_cast<cplx *>(smem_raw) + (size_t)rib * padded_lenE<E>(Hx);
    const cplx *src = inter + (size_t)row * Hx;
#pragma unroll
    for (int q = 0; q < E; q++) {
        const int k = j + q * T;
        s[padE<E>(k)] = live ? src[k] : mk(0, 0);
    }
    __syncthreads();
    cplx v[E];
#pragma unroll
    for (int q = 0; q < E; q++) {
        const int k = j + q * T;
        if (k == 0) {
            const cplx X = s[0]; // (DC, Nyquist), both real
            v[q] = mk(0.5 * (X.x + X.y), 0.5 * (X.x - X.y));
        } else {
            const cplx A = s[padE<E>(k)], B = cconj(s[padE<E>(Hx - k)]);
            const cplx Ev = mk(0.5 * (A.x + B.x), 0.5 * (A.y + B.y));
            cplx e = tw[(size_t)k * (g.Nt / g.Mx)]; e.y = -e.y; // exp(+2 pi i k/Mx)
            const cplx Od = cmul(mk(0.5 * (A.x - B.x), 0.5 * (A.y - B.y)), e);
            v[q] = mk(Ev.x - Od.y, Ev.y + Od.x); // E + i O
        }
    }
    fft_blockE<1, E, LOG2N_CT>(v, s, g.log2Hx, j, tw, g.Nt);
    if (!live) return;
    // background polynomial of this row: B(x) = sum_p cx[p] xt^p, cx[p] = sum_q b_(p,q) yt^q
    double cx[MAX_DEG + 1];
#pragma unroll
    for (int p = 0; p <= MAX_DEG; p++) cx[p] = 0.0;
    {
        const double yt = (2.0 * row + 1.0 - g.ny) / (double)g.ny;
        const double *b = coef + (size_t)g.NK * g.L * g.L;
        for (int sI = 0; sI < g.NB; sI++) {
            double yp = 1.0;
            for (int k = 0; k < g.pj[sI]; k++) yp *= yt;
#pragma unroll
            for (int p = 0; p <= MAX_DEG; p++) if (g.pi[sI] == p) cx[p] = fma(b[sI], yp, cx[p]);
        }
    }
    // mode 1 (plain convolution, f2): D = +M; the science image is not read and there is no background (NB = 0)
    const double scale = (mode ? -1.0 : 1.0) / ((double)Hx * (double)g.My), inx = 1.0 / (double)g.nx;
    const size_t ro = (size_t)row * g.nx;
    const bool vec = ((g.nx & 1) == 0) && (((size_t)S | (size_t)D) & 15) == 0;
#pragma unroll
    for (int q = 0; q < E; q++) {
        const int x0 = 2 * (j + q * T);
        if (x0 >= g.nx) continue;
        const double xa = (2.0 * x0 + 1.0 - g.nx) * inx, xb = (2.0 * x0 + 3.0 - g.nx) * inx;
        const double ba = fma(fma(fma(cx[3], xa, cx[2]), xa, cx[1]), xa, cx[0]);
        const double bb = fma(fma(fma(cx[3], xb, cx[2]), xb, cx[1]), xb, cx[0]);
        if (vec) {
            const double2 sv = mode ? make_double2(0.0, 0.0) : *reinterpret_cast<const double2 *>(S + ro + x0);
            double2 o; o.x = sv.x - scale * v[q].x - ba; o.y = sv.y - scale * v[q].y - bb;
            *reinterpret_cast<double2 *>(D + ro + x0) = o;
        } else {
            D[ro + x0] = (mode ? 0.0 : S[ro + x0]) - scale * v[q].x - ba;
            if (x0 + 1 < g.nx) D[ro + x0 + 1] = (mode ? 0.0 : S[ro + x0 + 1]) - scale * v[q].y - bb;
        }
    }
}

// One thread per border pixel (within w of an edge).  For every tap (u,v) whose source pixel
// (x-u, y-v) leaves the frame, the padded-grid FFT used Rpad((x-u) mod Mx, (y-v) mod My) (zero in
// the padding) where the method wants R((x-u) mod nx, (y-v) mod ny): subtract the difference.
__global__ void __launch_bounds__(128) wrapfix_kernel(const double *__restrict__ R, const double *__restrict__ coef,
                                                     double *__restrict__ D, Geom g, int mode) {
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
    if (live && part == 0) D[(size_t)y * nx + x] -= mode ? -corr : corr;
}

int col_cfg(const Geom &g, int *threads, size_t *smem); // sfft_fwd.cu
int row_cfg(const Geom &g, int E, int *threads, size_t *smem);
int fft_E(const char *env, int N, int dflt);

cudaError_t launch_subtract(sfft_plan *p, const double *S, const double *R, const double *coef, double *D,
                            const cplx *spec, int mode) {
    const Geom &g = p->g;
    if (!spec) spec = p->specTo;
    cudaStream_t st = p->stream;
    const bool pipe = colpipe_ok(g);
    if (!pipe) { KLaunch kl(p, "ktab"); ktab_kernel<<<dim3((g.Hx + 1 + 127) / 128, g.w + 1, g.NK), 128, 0, st>>>(coef, p->E, g, p->tw); }
    int threads; size_t smem;
    const int C = col_cfg(g, &threads, &smem);
    smem += (size_t)g.NK * g.L * (C + 1) * sizeof(cplx);
    static bool attr_set = false;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(col_inv_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 220 * 1024);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(row_inv_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(row_inv_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(row_inv_kernel<8, 11>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    if (pipe) { cudaError_t e = launch_colpipe_inv(p, spec, coef, p->inter); if (e != cudaSuccess) return e; }
    else { KLaunch kl(p, "col_inv"); col_inv_kernel<<<g.Hx / C, threads, smem, st>>>(spec, p->E, p->inter, C, g, p->tw); }
    const int ER = fft_E("SFFT_ROW_E", g.Hx, 8);
    int rthreads; size_t rsmem;
    const int RPB = row_cfg(g, ER, &rthreads, &rsmem);
    {
        KLaunch kl(p, "row_inv");
        if (ER == 8 && g.log2Hx == 11 && RPB == 1) row_inv_kernel<8, 11><<<g.ny, rthreads, rsmem, st>>>(p->inter, S, coef, D, g, p->tw, mode);
        else if (ER == 8) row_inv_kernel<8><<<(g.ny + RPB - 1) / RPB, rthreads, rsmem, st>>>(p->inter, S, coef, D, g, p->tw, mode);
        else row_inv_kernel<16><<<(g.ny + RPB - 1) / RPB, rthreads, rsmem, st>>>(p->inter, S, coef, D, g, p->tw, mode);
    }
    if ((g.Mx != g.nx || g.My != g.ny) && g.w > 0) {
        const long long nb = 2LL * g.w * g.nx + 2LL * g.w * (g.ny - 2 * g.w);
        KLaunch kl(p, "wrapfix");
        wrapfix_kernel<<<(unsigned)((4 * nb + 127) / 128), 128, 0, st>>>(R, coef, D, g, mode);
    }
    return cudaGetLastError();
}

} // namespace sfft
