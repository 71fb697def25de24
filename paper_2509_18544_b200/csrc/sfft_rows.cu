// sfft_rows.cu -- the row passes of the 2-D FFTs (steps a1 and a5; BASELINE.json north_star (a), (d); SURVEY.md
// 8(a) rows a1, a5).
//
// A row of Mx reals (the frame's nx pixels, zero-padded) is transformed as Hx = Mx/2 complex numbers
// z[n] = x[2n] + i x[2n+1] and untangled to the half spectrum kx = 0..Hx, stored as Hx columns with column 0
// = X[0] + i X[Hx] (both real).  Two adjacent image rows are transformed TOGETHER, one per lane parity
// (lane 2j + r works on row y0 + r): with the column-major planes (sfft_fft.cuh) the two rows' values of one kx
// are then one whole 32-byte sector per lane pair -- the piece size at which scattered stores and loads still
// run at > 70 % of the HBM rate on B200 (16-byte pieces: 17 %).
//
// T = Hx/16 threads per row, 16 complex values per thread.  Forward passes: radix 16, radix Hx/128, radix 8.
// In the last pass a thread takes the two butterflies A = j and B = Hx/8 - j, whose outputs Z[A + m Hx/8] and
// Z[B + (7-m) Hx/8] are exactly the partners k <-> Hx - k of the real<->complex untangle: it happens in
// registers, without the extra shared-memory round trip of a separate untangle step (the row passes were bound
// by the shared-memory pipe: profiles/r01l_ncu_summary.md).  The inverse kernel mirrors this: tangle in
// registers, then radix 8 (butterflies A, B), radix Hx/128, radix 16, and the fused D = S - M - B.
#include "sfft_internal.h"

namespace sfft {

constexpr int ROW_THREADS = 256;

template <int LOG2H> struct RowCfg {
    static constexpr int Hx = 1 << LOG2H, T = Hx / 16, GT = 2 * T, RP = ROW_THREADS / GT;
    static constexpr int R2 = Hx / 128;                       // middle radix: 4, 8 or 16
    static constexpr size_t SMEM = (size_t)RP * 2 * Hx * sizeof(cplx);
};

__device__ __forceinline__ double ipow_small(double b, int e) {
    double r = 1.0;
    for (int k = 0; k < e; k++) r *= b;
    return r;
}

// exp(-2 pi i m/16), m = 0..7
__device__ __forceinline__ cplx w16(int m) {
    switch (m) {
    case 0: return mk(1.0, 0.0);
    case 1: return mk(SFFT_C1, -SFFT_S1);
    case 2: return mk(SFFT_R2, -SFFT_R2);
    case 3: return mk(SFFT_S1, -SFFT_C1);
    case 4: return mk(0.0, -1.0);
    case 5: return mk(-SFFT_S1, -SFFT_C1);
    case 6: return mk(-SFFT_R2, -SFFT_R2);
    default: return mk(-SFFT_C1, -SFFT_S1);
    }
}

// untangle of one partner pair: ZA = Z[k], ZB = Z[Hx - k], u = exp(-2 pi i k/Mx):
//   X[k] = E + u O,  X[Hx - k] = conj(E - u O),  E = (ZA + conj ZB)/2,  O = (ZA - conj ZB)/(2i)
__device__ __forceinline__ void untangle(cplx ZA, cplx ZB, cplx u, cplx &Xk, cplx &Xnk) {
    const cplx E = mk(0.5 * (ZA.x + ZB.x), 0.5 * (ZA.y - ZB.y));
    const cplx O = mk(0.5 * (ZA.y + ZB.y), -0.5 * (ZA.x - ZB.x));
    const cplx P = cmul(u, O);
    Xk = mk(E.x + P.x, E.y + P.y);
    Xnk = mk(E.x - P.x, -(E.y - P.y));
}
// the inverse: XA = X[k], XB = X[Hx - k]:  Z[k] = Ev + i Od,  Z[Hx - k] = conj(Ev - i Od),
//   Ev = (XA + conj XB)/2,  Od = (XA - conj XB)/2 * conj(u)
__device__ __forceinline__ void tangle(cplx XA, cplx XB, cplx u, cplx &Zk, cplx &Znk) {
    const cplx Ev = mk(0.5 * (XA.x + XB.x), 0.5 * (XA.y - XB.y));
    const cplx Od = cmul(mk(0.5 * (XA.x - XB.x), 0.5 * (XA.y + XB.y)), cconj(u));
    Zk = mk(Ev.x - Od.y, Ev.y + Od.x);
    Znk = mk(Ev.x + Od.y, Od.x - Ev.y);
}

// ------------------------------------------------------------------------------------------ forward
// rows: img (ny x nx real, optional mask) -> inter[i] (Hx columns x My, column-major), i = 0..NI-1, weights xt^i;
// also row moments mu[m][y] = sum_x xt^m (m.img), m = 0..NMOM-1 (for Gamma / Delta).
// grid = ceil(ny / (2 RP)); block 256 = RP row pairs of 2 T threads; dynamic smem RowCfg::SMEM
template <int LOG2H>
__global__ void __launch_bounds__(ROW_THREADS, 2)
row_fwd_kernel(const double *__restrict__ img, const uint8_t *__restrict__ mask, cplx *__restrict__ inter, int NI,
               double *__restrict__ mu, int NMOM, Geom g, const cplx *__restrict__ tw) {
    using C = RowCfg<LOG2H>;
    constexpr int Hx = C::Hx, T = C::T, GT = C::GT, TP = 2 * T; // TP = Hx/8: butterflies of the last pass
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ double wpart[ROW_THREADS / 32][2][8];
    const int grp = threadIdx.x / GT, t = threadIdx.x - grp * GT, r = t & 1, j = t >> 1, bar_id = 1 + grp;
    cplx *X = reinterpret_cast<cplx *>(smem_raw) + (size_t)grp * 2 * Hx;
    const int y = (blockIdx.x * C::RP + grp) * 2 + r, nx = g.nx, ny = g.ny, My = g.My, Nt = g.Nt;
    const bool live = y < ny;
    const double inv_nx = 1.0 / (double)nx;
    const size_t rowoff = (size_t)y * nx;
    const bool vec = ((nx & 1) == 0) && (((size_t)img & 15) == 0);
    const int A = j, B = j == 0 ? T : TP - j;
    const cplx wA = tw[(size_t)A * (Nt >> LOG2H)], wB = tw[(size_t)B * (Nt >> LOG2H)]; // exp(-2 pi i jb/Hx)
    const cplx uA = tw[(size_t)A * (Nt >> (LOG2H + 1))], uT = tw[(size_t)T * (Nt >> (LOG2H + 1))]; // exp(-2 pi i k/Mx)

    for (int i = 0; i < NI; i++) {
        cplx v[16];
        double mom[8];
#pragma unroll
        for (int m = 0; m < 8; m++) mom[m] = 0.0;
#pragma unroll
        for (int q = 0; q < 16; q++) {
            const int x0 = 2 * (j + q * T);
            double a = 0.0, b = 0.0;
            if (live) {
                if (vec) { // even nx, 16-byte aligned image: one 16-byte load per pixel pair
                    if (x0 < nx) { const double2 ab = *reinterpret_cast<const double2 *>(img + rowoff + x0); a = ab.x; b = ab.y; }
                } else {
                    if (x0 < nx) a = img[rowoff + x0];
                    if (x0 + 1 < nx) b = img[rowoff + x0 + 1];
                }
                if (mask) {
                    if (x0 < nx && !mask[rowoff + x0]) a = 0.0;
                    if (x0 + 1 < nx && !mask[rowoff + x0 + 1]) b = 0.0;
                }
            }
            const double xa = (2.0 * x0 + 1.0 - nx) * inv_nx, xb = (2.0 * x0 + 3.0 - nx) * inv_nx;
            if (i == 0 && NMOM > 0) {
                double pa = a, pb = b;
#pragma unroll
                for (int m = 0; m < 8; m++)
                    if (m < NMOM) { mom[m] += pa + pb; pa *= xa; pb *= xb; }
            }
            v[q] = mk(a * ipow_small(xa, i), b * ipow_small(xb, i));
        }
        if (i == 0 && NMOM > 0) {
            // deterministic reduction over the T threads of each row: lanes of equal parity inside a warp, then warps
#pragma unroll
            for (int m = 0; m < 8; m++)
                if (m < NMOM)
#pragma unroll
                    for (int off = 16; off >= 2; off >>= 1) mom[m] += __shfl_xor_sync(0xffffffffu, mom[m], off);
            const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
            if (lane < 2) {
#pragma unroll
                for (int m = 0; m < 8; m++) // static indices: a run-time bound here would push mom[] into local memory
                    if (m < NMOM) wpart[wid][lane][m] = mom[m];
            }
            group_sync(bar_id, GT);
            if (j == 0 && live) {
                const int w0 = (grp * GT) >> 5, nwarp = GT >> 5;
                for (int m = 0; m < NMOM; m++) {
                    double acc = 0.0;
                    for (int k = 0; k < nwarp; k++) acc += wpart[w0 + k][r][m];
                    mu[(size_t)m * ny + y] = acc;
                }
            }
        }
        group_sync(bar_id, GT); // the previous transform's last-pass reads of X are done
        {   // pass 1: radix 16, no twiddles
            dft16<-1>(v);
#pragma unroll
            for (int m = 0; m < 16; m++) X[(size_t)out_pos<16, 4>(j, m, 0) * 2 + r] = v[m];
        }
        group_sync(bar_id, GT);
        load_canonical<4, 2>(v, X, r, j, T);
        group_sync(bar_id, GT);
        pass_store<C::R2, -1, 4, 2>(v, X, r, j, T, 4, tw, Nt);
        group_sync(bar_id, GT);
        // last pass: radix 8, Ns = Hx/8, butterflies A and B
        cplx zA[8], zB[8];
#pragma unroll
        for (int m = 0; m < 8; m++) {
            zA[m] = X[(size_t)swz<4>(A + m * TP) * 2 + r];
            zB[m] = X[(size_t)swz<4>(B + m * TP) * 2 + r];
        }
        bfly_w<8, -1>(zA, wA);
        bfly_w<8, -1>(zB, wB);
        cplx *dst = inter + (size_t)i * Hx * My + y;
        if (j != 0) {
#pragma unroll
            for (int m = 0; m < 8; m++) {
                cplx Xk, Xnk;
                untangle(zA[m], zB[7 - m], cmul(uA, w16(m)), Xk, Xnk);
                if (live) { dst[(size_t)(A + m * TP) * My] = Xk; dst[(size_t)(B + (7 - m) * TP) * My] = Xnk; }
            }
        } else {
            // butterfly 0 pairs with itself (k = m Hx/8 <-> (8-m) Hx/8; k = 0 is the packed DC/Nyquist pair), and so
            // does butterfly T (k = T + m Hx/8 <-> T + (7-m) Hx/8)
            if (live) dst[0] = mk(zA[0].x + zA[0].y, zA[0].x - zA[0].y);
#pragma unroll
            for (int m = 1; m <= 4; m++) {
                cplx Xk, Xnk;
                untangle(zA[m], zA[8 - m], w16(m), Xk, Xnk);
                if (live) { dst[(size_t)(m * TP) * My] = Xk; if (m < 4) dst[(size_t)((8 - m) * TP) * My] = Xnk; }
            }
#pragma unroll
            for (int m = 0; m < 4; m++) {
                cplx Xk, Xnk;
                untangle(zB[m], zB[7 - m], cmul(uT, w16(m)), Xk, Xnk);
                if (live) { dst[(size_t)(T + m * TP) * My] = Xk; dst[(size_t)(T + (7 - m) * TP) * My] = Xnk; }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------ inverse
// inter (Hx columns x My, column-major) -> D = S - M - B (mode 0) or D = +M (mode 1: plain convolution, f2)
template <int LOG2H>
__global__ void __launch_bounds__(ROW_THREADS, 2)
row_inv_kernel(const cplx *__restrict__ inter, const double *__restrict__ S, const double *__restrict__ coef,
               double *__restrict__ D, Geom g, const cplx *__restrict__ tw, int mode) {
    using C = RowCfg<LOG2H>;
    constexpr int Hx = C::Hx, T = C::T, GT = C::GT, TP = 2 * T;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int grp = threadIdx.x / GT, t = threadIdx.x - grp * GT, r = t & 1, j = t >> 1, bar_id = 1 + grp;
    cplx *X = reinterpret_cast<cplx *>(smem_raw) + (size_t)grp * 2 * Hx;
    const int y = (blockIdx.x * C::RP + grp) * 2 + r, nx = g.nx, ny = g.ny, My = g.My, Nt = g.Nt;
    const bool live = y < ny;
    const int A = j, B = j == 0 ? T : TP - j;
    const cplx uA = tw[(size_t)A * (Nt >> (LOG2H + 1))], uT = tw[(size_t)T * (Nt >> (LOG2H + 1))];
    const cplx *src = inter + y;
    cplx zA[8], zB[8];
    {
        cplx xA[8], xB[8];
#pragma unroll
        for (int m = 0; m < 8; m++) {
            xA[m] = live ? src[(size_t)(A + m * TP) * My] : mk(0.0, 0.0);
            xB[m] = live ? src[(size_t)(B + m * TP) * My] : mk(0.0, 0.0);
        }
        if (j != 0) {
#pragma unroll
            for (int m = 0; m < 8; m++) tangle(xA[m], xB[7 - m], cmul(uA, w16(m)), zA[m], zB[7 - m]);
        } else {
            zA[0] = mk(0.5 * (xA[0].x + xA[0].y), 0.5 * (xA[0].x - xA[0].y)); // (DC, Nyquist), both real
#pragma unroll
            for (int m = 1; m <= 4; m++) {
                cplx Zk, Znk;
                tangle(xA[m], xA[8 - m], w16(m), Zk, Znk);
                zA[m] = Zk;
                if (m < 4) zA[8 - m] = Znk;
            }
#pragma unroll
            for (int m = 0; m < 4; m++) tangle(xB[m], xB[7 - m], cmul(uT, w16(m)), zB[m], zB[7 - m]);
        }
    }
    // pass 1: radix 8, no twiddles, butterflies A and B
    dft8<1>(zA);
    dft8<1>(zB);
#pragma unroll
    for (int m = 0; m < 8; m++) {
        X[(size_t)out_pos<8, 3>(A, m, 0) * 2 + r] = zA[m];
        X[(size_t)out_pos<8, 3>(B, m, 0) * 2 + r] = zB[m];
    }
    group_sync(bar_id, GT);
    cplx v[16];
    load_canonical<3, 2>(v, X, r, j, T);
    group_sync(bar_id, GT);
    pass_store<C::R2, 1, 3, 2>(v, X, r, j, T, 3, tw, Nt);
    group_sync(bar_id, GT);
    load_canonical<3, 2>(v, X, r, j, T);
    pass_regs<16, 1>(v, j, T, LOG2H - 4, tw, Nt);
    if (!live) return;
    // background polynomial of this row: B(x) = sum_p cx[p] xt^p, cx[p] = sum_q b_(p,q) yt^q
    double cx[MAX_DEG + 1];
#pragma unroll
    for (int p = 0; p <= MAX_DEG; p++) cx[p] = 0.0;
    {
        const double yt = (2.0 * y + 1.0 - ny) / (double)ny;
        const double *b = coef + (size_t)g.NK * g.L * g.L;
        for (int sI = 0; sI < g.NB; sI++) {
            double yp = 1.0;
            for (int k = 0; k < g.pj[sI]; k++) yp *= yt;
#pragma unroll
            for (int p = 0; p <= MAX_DEG; p++) if (g.pi[sI] == p) cx[p] = fma(b[sI], yp, cx[p]);
        }
    }
    // mode 1 (plain convolution, f2): D = +M; the science image is not read and there is no background (NB = 0)
    const double scale = (mode ? -1.0 : 1.0) / ((double)Hx * (double)My), inx = 1.0 / (double)nx;
    const size_t ro = (size_t)y * nx;
    const bool vec = ((nx & 1) == 0) && (((size_t)S | (size_t)D) & 15) == 0;
#pragma unroll
    for (int q = 0; q < 16; q++) {
        const int x0 = 2 * (j + q * T);
        if (x0 >= nx) continue;
        const double xa = (2.0 * x0 + 1.0 - nx) * inx, xb = (2.0 * x0 + 3.0 - nx) * inx;
        const double ba = fma(fma(fma(cx[3], xa, cx[2]), xa, cx[1]), xa, cx[0]);
        const double bb = fma(fma(fma(cx[3], xb, cx[2]), xb, cx[1]), xb, cx[0]);
        if (vec) {
            const double2 sv = mode ? make_double2(0.0, 0.0) : *reinterpret_cast<const double2 *>(S + ro + x0);
            double2 o; o.x = sv.x - scale * v[q].x - ba; o.y = sv.y - scale * v[q].y - bb;
            *reinterpret_cast<double2 *>(D + ro + x0) = o;
        } else {
            D[ro + x0] = (mode ? 0.0 : S[ro + x0]) - scale * v[q].x - ba;
            if (x0 + 1 < nx) D[ro + x0 + 1] = (mode ? 0.0 : S[ro + x0 + 1]) - scale * v[q].y - bb;
        }
    }
}

// ------------------------------------------------------------------------------------------ host side
template <int LOG2H> static cudaError_t rows_attr() {
    cudaError_t e = cudaFuncSetAttribute(row_fwd_kernel<LOG2H>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RowCfg<LOG2H>::SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(row_inv_kernel<LOG2H>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RowCfg<LOG2H>::SMEM);
    return e;
}
cudaError_t rows_init() { // per device, at plan creation
    cudaError_t e = rows_attr<9>();
    if (e == cudaSuccess) e = rows_attr<10>();
    if (e == cudaSuccess) e = rows_attr<11>();
    return e;
}

cudaError_t launch_row_fwd(sfft_plan *p, const double *img, const uint8_t *mask, cplx *inter, int NI, double *mu, int NMOM) {
    const Geom &g = p->g;
    KLaunch kl(p, NI > 1 ? "row_fwd_R" : "row_fwd_S");
    switch (g.log2Hx) {
    case 9: row_fwd_kernel<9><<<(g.ny + 2 * RowCfg<9>::RP - 1) / (2 * RowCfg<9>::RP), ROW_THREADS, RowCfg<9>::SMEM, p->stream>>>(img, mask, inter, NI, mu, NMOM, g, p->tw); break;
    case 10: row_fwd_kernel<10><<<(g.ny + 2 * RowCfg<10>::RP - 1) / (2 * RowCfg<10>::RP), ROW_THREADS, RowCfg<10>::SMEM, p->stream>>>(img, mask, inter, NI, mu, NMOM, g, p->tw); break;
    case 11: row_fwd_kernel<11><<<(g.ny + 2 * RowCfg<11>::RP - 1) / (2 * RowCfg<11>::RP), ROW_THREADS, RowCfg<11>::SMEM, p->stream>>>(img, mask, inter, NI, mu, NMOM, g, p->tw); break;
    default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

cudaError_t launch_row_inv(sfft_plan *p, const cplx *inter, const double *S, const double *coef, double *D, int mode) {
    const Geom &g = p->g;
    KLaunch kl(p, "row_inv");
    switch (g.log2Hx) {
    case 9: row_inv_kernel<9><<<(g.ny + 2 * RowCfg<9>::RP - 1) / (2 * RowCfg<9>::RP), ROW_THREADS, RowCfg<9>::SMEM, p->stream>>>(inter, S, coef, D, g, p->tw, mode); break;
    case 10: row_inv_kernel<10><<<(g.ny + 2 * RowCfg<10>::RP - 1) / (2 * RowCfg<10>::RP), ROW_THREADS, RowCfg<10>::SMEM, p->stream>>>(inter, S, coef, D, g, p->tw, mode); break;
    case 11: row_inv_kernel<11><<<(g.ny + 2 * RowCfg<11>::RP - 1) / (2 * RowCfg<11>::RP), ROW_THREADS, RowCfg<11>::SMEM, p->stream>>>(inter, S, coef, D, g, p->tw, mode); break;
    default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

} // namespace sfft
