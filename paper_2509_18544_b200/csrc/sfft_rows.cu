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
#include <cuda.h>
#include <new>
#include <type_traits>
#include "sfft_internal.h"

namespace sfft {

constexpr int ROW_THREADS = 256;

constexpr int ROW_RING = 3;

// A WORKER is the group of 2 T threads of one row pair; a CTA holds RP = 256 / (2 T) workers, two CTAs share an SM.
// Workers are persistent: they loop over row pairs, and the input of the next steps is in flight (bulk copies
// completing on mbarriers, one elected thread) while the current pair is transformed.
template <int LOG2H> struct RowCfg {
    static constexpr int Hx = 1 << LOG2H, T = Hx / 16, GT = 2 * T, RP = ROW_THREADS / GT;
    static constexpr int R2 = Hx / 128;                       // middle radix: 4, 8 or 16
    static constexpr int QP = 8 * T;                          // pixels of a quarter row (Mx / 4)
    static constexpr int FSLOT = 2 * QP + 16;                 // forward ring slot in doubles: two quarter rows, the second
                                                              // skewed by 64 B (+ pad to 128 B) against bank conflicts
    static constexpr size_t XBYTES = (size_t)RP * 2 * Hx * sizeof(cplx);
    static constexpr size_t SMEM_F = XBYTES + (size_t)RP * ROW_RING * FSLOT * sizeof(double);
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
// grid: persistent, <= 2 CTAs per SM; block 256 = RP workers of 2 T threads; dynamic smem RowCfg::SMEM_F.
// BULK (even nx, 16-byte aligned image): the two rows arrive quarter by quarter through a 3-slot ring of bulk copies
// (every weight i re-reads the pair from L2); otherwise plain loads.
template <int LOG2H, bool BULK, bool MASK>
__global__ void __launch_bounds__(ROW_THREADS, 2)
row_fwd_kernel(const double *__restrict__ img, const uint8_t *__restrict__ mask, cplx *__restrict__ inter, int NI,
               double *__restrict__ mu, int NMOM, Geom g, const cplx *__restrict__ tw, const cplx *__restrict__ rtw) {
    using C = RowCfg<LOG2H>;
    constexpr int Hx = C::Hx, T = C::T, GT = C::GT, TP = 2 * T, QP = C::QP; // TP = Hx/8: butterflies of the last pass
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ unsigned long long full[C::RP * ROW_RING], done[C::RP * ROW_RING];
    const int grp = threadIdx.x / GT, t = threadIdx.x - grp * GT, r = t & 1, j = t >> 1, bar_id = 1 + grp;
    cplx *X = reinterpret_cast<cplx *>(smem_raw) + (size_t)grp * 2 * Hx;
    // warp partials of the row moments [warp of the worker][row][m]: they live in the exchange buffer, which is idle
    // during the load phase (two CTAs per SM leave no room for another static array)
    double (*wpart)[2][8] = reinterpret_cast<double (*)[2][8]>(X);
    double *ring = reinterpret_cast<double *>(smem_raw + C::XBYTES) + (size_t)grp * ROW_RING * C::FSLOT;
    unsigned long long *bar = full + grp * ROW_RING, *rel = done + grp * ROW_RING;
    if (BULK && t == 0) {
        for (int k = 0; k < ROW_RING; k++) { mbar_init(&bar[k], 1); mbar_init(&rel[k], GT); }
        mbar_fence_init();
    }
    __syncthreads();
    const int nx = g.nx, ny = g.ny, My = g.My, Nt = g.Nt, npairs = (ny + 1) >> 1;
    const int wid = blockIdx.x * C::RP + grp, nw = gridDim.x * C::RP;
    const int nmine = wid < npairs ? (npairs - wid + nw - 1) / nw : 0;
    const int nitems = nmine * NI, nsteps = nitems * 4;
    const double inv_nx = 1.0 / (double)nx;
    auto issue = [&](int s) { // one thread: quarter Q of both rows of item n into slot s % RING
        const int n = s >> 2, Q = s & 3, slot = s % ROW_RING;
        const int y0 = 2 * (wid + (n / NI) * nw);
        int px = nx - Q * QP; px = px < 0 ? 0 : (px > QP ? QP : px);
        const unsigned bytes = (unsigned)px * 8u;
        const bool two = y0 + 1 < ny;
        mbar_expect(&bar[slot], two ? 2u * bytes : bytes);
        if (bytes) {
            double *dst = ring + (size_t)slot * C::FSLOT;
            const double *src = img + (size_t)y0 * nx + Q * QP;
            bulk_g2s(dst, src, bytes, &bar[slot]);
            if (two) bulk_g2s(dst + QP + 8, src + nx, bytes, &bar[slot]);
        }
    };
    if (BULK && t == 0)
        for (int s = 0; s < ROW_RING && s < nsteps; s++) issue(s);

    int s = 0;
    const int j_outer_ = j; // (see the note at opaque_index)
    for (int n = 0; n < nitems; n++) {
        const int j = opaque_index(j_outer_);
        // xt of the thread's pixel pairs: pixel 2 (j + q T) has xt = xa0 + q xstep, its neighbour xt + xpix
        const double xa0 = (4.0 * j + 1.0 - nx) * inv_nx, xstep = 4.0 * T * inv_nx, xpix = 2.0 * inv_nx;
        const int A = j, B = j == 0 ? T : TP - j;
        const int i = n % NI, y = 2 * (wid + (n / NI) * nw) + r;
        const bool live = y < ny;
        const size_t rowoff = (size_t)y * nx;
        cplx v[16];
        // weight xt^i as the one-hot cubic c0 + x (c1 + x (c2 + x c3)): three fused multiply-adds, no branches on i
        const double c0 = i == 0 ? 1.0 : 0.0, c1 = i == 1 ? 1.0 : 0.0, c2 = i == 2 ? 1.0 : 0.0, c3 = i == 3 ? 1.0 : 0.0;
        // the load phase; NM = number of row moments accumulated beside it (0: none; the instances 3, 5, 8 cover
        // NMOM <= 3, <= 5, <= 7 -- their accumulators live only in the instance that needs them)
        auto load = [&](auto nm_tag) {
            constexpr int NM = decltype(nm_tag)::value;
            double mom[NM > 0 ? NM : 1];
#pragma unroll
            for (int m = 0; m < (NM > 0 ? NM : 1); m++) mom[m] = 0.0;
#pragma unroll
            for (int Q = 0; Q < 4; Q++) {
                const int slot = s % ROW_RING;
                if (BULK) mbar_wait(&bar[slot], (unsigned)(s / ROW_RING) & 1u);
#pragma unroll
                for (int qq = 0; qq < 4; qq++) {
                    const int q = 4 * Q + qq, x0 = 2 * (j + q * T);
                    double a = 0.0, b = 0.0;
                    if (BULK) {
                        const double2 ab = *reinterpret_cast<const double2 *>(ring + (size_t)slot * C::FSLOT + r * (QP + 8) + 2 * j + 2 * T * qq);
                        if (live && x0 < nx) { a = ab.x; b = ab.y; }
                    } else if (live) {
                        if (x0 < nx) a = img[rowoff + x0];
                        if (x0 + 1 < nx) b = img[rowoff + x0 + 1];
                    }
                    if (MASK && live) {
                        if (x0 < nx && !mask[rowoff + x0]) a = 0.0;
                        if (x0 + 1 < nx && !mask[rowoff + x0 + 1]) b = 0.0;
                    }
                    const double xa = fma((double)q, xstep, xa0), xb = xa + xpix; // xt of pixels x0, x0 + 1
                    if (NM > 0) {
                        double pa = a, pb = b;
#pragma unroll
                        for (int m = 0; m < NM; m++) { mom[m] += pa + pb; pa *= xa; pb *= xb; }
                    }
                    v[q] = mk(a * fma(xa, fma(xa, fma(xa, c3, c2), c1), c0), b * fma(xb, fma(xb, fma(xb, c3, c2), c1), c0));
                }
                if (BULK) {
                    // release the slot: every thread arrives (release semantics: its loads of the slot are done) and the
                    // issuing thread refills it once all have.  (A bar.sync is not enough here: the copy engine is not
                    // ordered behind it -- a refill could overtake a slow warp's reads.)
                    slot_release(&rel[slot]);
                    if (t == 0 && s + ROW_RING < nsteps) { mbar_wait(&rel[slot], (unsigned)(s / ROW_RING) & 1u); issue(s + ROW_RING); }
                    s++;
                }
            }
            if (NM > 0) {
                // deterministic reduction over the T threads of each row: lanes of equal parity inside a warp, then warps
                group_sync(bar_id, GT); // the previous item's last-pass reads of X are done (wpart lives in X)
                const int lane = threadIdx.x & 31, wrp = t >> 5;
#pragma unroll
                for (int m = 0; m < NM; m++) {
#pragma unroll
                    for (int off = 16; off >= 2; off >>= 1) mom[m] += __shfl_xor_sync(0xffffffffu, mom[m], off);
                    if (lane < 2) wpart[wrp][lane][m] = mom[m];
                }
            }
        };
        if (i == 0 && NMOM > 0) {
            if (NMOM <= 3) load(std::integral_constant<int, 3>());
            else if (NMOM <= 5) load(std::integral_constant<int, 5>());
            else load(std::integral_constant<int, 8>());
            group_sync(bar_id, GT);
            if (j == 0 && live) {
                const int nwarp = GT >> 5;
                for (int m = 0; m < NMOM; m++) {
                    double acc = 0.0;
                    for (int k = 0; k < nwarp; k++) acc += wpart[k][r][m];
                    mu[(size_t)m * ny + y] = acc;
                }
            }
        } else load(std::integral_constant<int, 0>());
        group_sync(bar_id, GT); // the previous transform's last-pass reads of X (and of wpart) are done
        {   // pass 1: radix 16, no twiddles
            dft16<-1>(v);
#pragma unroll
            for (int m = 0; m < 16; m++) X[(size_t)out_pos<16, 4>(j, m, 0) * 2 + r] = v[m];
        }
        group_sync(bar_id, GT);
        load_canonical<4, 2>(v, X, r, j, T);
        group_sync(bar_id, GT);
        pass_store<C::R2, -1, 4, 2>(v, X, r, j, T, 4, tw, Nt);
        // twiddles of the last pass and of the untangle: fetched here (not kept across the passes: 16 registers), their
        // latency hides behind the barrier
        // (from the compact table rtw[3][T]: three coalesced loads.  Gathered from the big table they were 16 lines per warp
        // and load; with the shared-memory carve-out at its maximum the L1 is ~30 KB, every one missed, item after item,
        // and the butterflies below waited for L2: 16 % of the kernel's stall samples)
        const cplx wA = rtw[j], wB = rtw[T + j]; // exp(-2 pi i jb/Hx), jb = A, B
        const cplx uA = rtw[2 * T + j];          // exp(-2 pi i k/Mx), k = A (thread 0: T)
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
                untangle(zB[m], zB[7 - m], cmul(uA, w16(m)), Xk, Xnk);
                if (live) { dst[(size_t)(T + m * TP) * My] = Xk; dst[(size_t)(T + (7 - m) * TP) * My] = Xnk; }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------ inverse
__device__ __forceinline__ void l2_prefetch(const void *gsrc, unsigned bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(gsrc), "r"(bytes) : "memory");
}

__device__ __forceinline__ void tma_prefetch2(const CUtensorMap *tm, int c0, int c1) {
    asm volatile("cp.async.bulk.prefetch.tensor.2d.L2.global.tile [%0, {%1, %2}];" ::"l"(tm), "r"(c0), "r"(c1) : "memory");
}

// inter (Hx columns x My, column-major; tensor map tmI: boxes {2 rows, Hx/8 kx} = the 32-byte sectors of one row
// pair) -> D = S - M - B (mode 0) or D = +M (mode 1: plain convolution, f2).
// A thread needs exactly 16 elements of the intermediate (its two butterflies) and nobody else needs them, so they
// go straight to registers: 16 independent 16-byte loads, lane pairs covering whole 32-byte sectors.  What hides
// their latency is a TMA PREFETCH: while a pair is transformed, one thread asks the copy engine to bring the next
// pair's boxes (and its two science rows) into L2 -- no shared-memory ring, no barriers, nothing to release.
// grid: persistent, <= 2 CTAs per SM; block 256 = RP workers of 2 T threads; dynamic smem RowCfg::XBYTES
template <int LOG2H>
__global__ void __launch_bounds__(ROW_THREADS, 2)
row_inv_kernel(const __grid_constant__ CUtensorMap tmI, const cplx *__restrict__ inter, const double *__restrict__ S,
               const double *__restrict__ coef, double *__restrict__ D, Geom g, const cplx *__restrict__ tw, int mode) {
    using C = RowCfg<LOG2H>;
    constexpr int Hx = C::Hx, T = C::T, GT = C::GT, TP = 2 * T;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int grp = threadIdx.x / GT, t = threadIdx.x - grp * GT, r = t & 1, j = t >> 1, bar_id = 1 + grp;
    cplx *X = reinterpret_cast<cplx *>(smem_raw) + (size_t)grp * 2 * Hx;
    const int nx = g.nx, ny = g.ny, My = g.My, Nt = g.Nt, npairs = (ny + 1) >> 1;
    const int wid = blockIdx.x * C::RP + grp, nw = gridDim.x * C::RP;
    const int nmine = wid < npairs ? (npairs - wid + nw - 1) / nw : 0;
    const int A = j, B = j == 0 ? T : TP - j;
    const bool vec = ((nx & 1) == 0) && (((size_t)S | (size_t)D) & 15) == 0;
    auto prefetch = [&](int n) { // one thread: the boxes and the science rows of row pair n towards L2
        const int y0 = 2 * (wid + n * nw);
#pragma unroll
        for (int m = 0; m < 8; m++) tma_prefetch2(&tmI, 2 * y0, m * TP);
        if (mode == 0 && vec) l2_prefetch(S + (size_t)y0 * nx, (unsigned)((y0 + 1 < ny ? 2 : 1) * nx * 8));
    };
    if (t == 0 && nmine > 0) prefetch(0);
    const cplx uA = tw[(size_t)(j == 0 ? T : A) * (Nt >> (LOG2H + 1))]; // exp(-2 pi i k/Mx), k = A (thread 0: T)
    const cplx wL = tw[(size_t)j * (Nt >> LOG2H)];                      // last pass: radix 16, Ns = T, one butterfly per thread
    const int j_outer_ = j; // (see the note at opaque_index)
    for (int n = 0; n < nmine; n++) {
        const int j = opaque_index(j_outer_);
        const int y = 2 * (wid + n * nw) + r;
        const bool live = y < ny;
        cplx zA[8], zB[8];
        {
            cplx xA[8], xB[8];
            const cplx *src = inter + y;
#pragma unroll
            for (int m = 0; m < 8; m++) {
                xA[m] = live ? src[(size_t)(A + m * TP) * My] : mk(0.0, 0.0);
                xB[m] = live ? src[(size_t)(B + m * TP) * My] : mk(0.0, 0.0);
            }
            if (t == 0 && n + 1 < nmine) prefetch(n + 1);
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
                for (int m = 0; m < 4; m++) tangle(xB[m], xB[7 - m], cmul(uA, w16(m)), zB[m], zB[7 - m]);
            }
        }
        // pass 1: radix 8, no twiddles, butterflies A and B
        dft8<1>(zA);
        dft8<1>(zB);
        group_sync(bar_id, GT); // the previous pair's last reads of X are done
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
        bfly_w<16, 1>(v, wL);
        if (!live) continue;
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
        if (vec) {
            // all loads of a batch first, then arithmetic and stores: one memory round trip per batch, not per pixel pair
#pragma unroll
            for (int h = 0; h < 4; h++) {
                double2 sv[4];
#pragma unroll
                for (int qq = 0; qq < 4; qq++) {
                    const int x0 = 2 * (j + (4 * h + qq) * T);
                    sv[qq] = (mode == 0 && x0 < nx) ? __ldcs(reinterpret_cast<const double2 *>(S + ro + x0)) : make_double2(0.0, 0.0);
                }
#pragma unroll
                for (int qq = 0; qq < 4; qq++) {
                    const int q = 4 * h + qq, x0 = 2 * (j + q * T);
                    const double xa = (2.0 * x0 + 1.0 - nx) * inx, xb = (2.0 * x0 + 3.0 - nx) * inx;
                    const double ba = fma(fma(fma(cx[3], xa, cx[2]), xa, cx[1]), xa, cx[0]);
                    const double bb = fma(fma(fma(cx[3], xb, cx[2]), xb, cx[1]), xb, cx[0]);
                    double2 o; o.x = sv[qq].x - scale * v[q].x - ba; o.y = sv[qq].y - scale * v[q].y - bb;
                    if (x0 < nx) __stcs(reinterpret_cast<double2 *>(D + ro + x0), o);
                }
            }
        } else {
#pragma unroll
            for (int q = 0; q < 16; q++) {
                const int x0 = 2 * (j + q * T);
                if (x0 >= nx) continue;
                const double xa = (2.0 * x0 + 1.0 - nx) * inx, xb = (2.0 * x0 + 3.0 - nx) * inx;
                const double ba = fma(fma(fma(cx[3], xa, cx[2]), xa, cx[1]), xa, cx[0]);
                const double bb = fma(fma(fma(cx[3], xb, cx[2]), xb, cx[1]), xb, cx[0]);
                D[ro + x0] = (mode ? 0.0 : S[ro + x0]) - scale * v[q].x - ba;
                if (x0 + 1 < nx) D[ro + x0 + 1] = (mode ? 0.0 : S[ro + x0 + 1]) - scale * v[q].y - bb;
            }
        }
    }
}

// ------------------------------------------------------------------------------------------ host side
template <int LOG2H> static cudaError_t rows_attr() {
    cudaError_t e = cudaFuncSetAttribute(row_fwd_kernel<LOG2H, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RowCfg<LOG2H>::SMEM_F);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(row_fwd_kernel<LOG2H, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RowCfg<LOG2H>::SMEM_F);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(row_fwd_kernel<LOG2H, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RowCfg<LOG2H>::SMEM_F);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(row_fwd_kernel<LOG2H, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RowCfg<LOG2H>::SMEM_F);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(row_inv_kernel<LOG2H>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RowCfg<LOG2H>::XBYTES);
    return e;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// rtw[0][j] = exp(-2 pi i j/Hx), rtw[1][j] = exp(-2 pi i B/Hx) (B = Hx/8 - j; j = 0: T), rtw[2][j] = exp(-2 pi i k/Mx)
// (k = j; j = 0: T), j < T = Hx/16: the last-pass and untangle twiddles of thread j of row_fwd_kernel, taken from tw
__global__ void rowtw_kernel(cplx *rtw, const cplx *__restrict__ tw, int T, int Nt, int Hx) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= T) return;
    const int TP = 2 * T, A = j, B = j == 0 ? T : TP - j;
    rtw[j] = tw[(size_t)A * (Nt / Hx)];
    rtw[T + j] = tw[(size_t)B * (Nt / Hx)];
    rtw[2 * T + j] = tw[(size_t)(j == 0 ? T : A) * (Nt / (2 * Hx))];
}

// per device and plan, at plan creation: kernel attributes and the tensor map of the a5 intermediate
// (plane [Hx][My] complex = [Hx][2 My] doubles, box {4 doubles = rows y0, y0+1 of one kx; Hx/8 kx})
cudaError_t rows_init(sfft_plan *p) {
    const Geom &g = p->g;
    cudaError_t e = rows_attr<9>();
    if (e == cudaSuccess) e = rows_attr<10>();
    if (e == cudaSuccess) e = rows_attr<11>();
    if (e != cudaSuccess) return e;
    {   // after twiddle_kernel (same stream)
        const int T = g.Hx / 16;
        e = cudaMalloc(&p->rtw, (size_t)3 * T * sizeof(cplx));
        if (e != cudaSuccess) return e;
        p->bytes += (size_t)3 * T * sizeof(cplx);
        rowtw_kernel<<<(T + 127) / 128, 128>>>(p->rtw, p->tw, T, g.Nt, g.Hx);
    }
    void *fn = nullptr; cudaDriverEntryPointQueryResult qr;
    e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr);
    if (e != cudaSuccess) return e;
    if (!fn || qr != cudaDriverEntryPointSuccess) return cudaErrorNotSupported;
    p->mapI = new (std::nothrow) CUtensorMap();
    if (!p->mapI) return cudaErrorMemoryAllocation;
    cuuint64_t dims[2] = {2 * (cuuint64_t)g.My, (cuuint64_t)g.Hx}, strides[1] = {(cuuint64_t)g.My * 16};
    cuuint32_t box[2] = {4, (cuuint32_t)(g.Hx / 8)}, es[2] = {1, 1};
    CUresult r = ((EncodeTiledFn)fn)(p->mapI, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, (void *)p->inter, dims, strides, box, es,
                                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}
void rows_free(sfft_plan *p) { delete p->mapI; p->mapI = nullptr; if (p->rtw) cudaFree(p->rtw); p->rtw = nullptr; }

template <int LOG2H> static int row_grid(const sfft_plan *p) {
    const int need = ((p->g.ny + 1) / 2 + RowCfg<LOG2H>::RP - 1) / RowCfg<LOG2H>::RP;
    int cap = 2 * p->sms;
    // while a factorisation runs beside us, leave a few SMs to it: persistent CTAs would otherwise block its chain of
    // small launches for the whole kernel
    if (p->factor_pending && cap > 2 * p->knob.factor_sms) cap -= 2 * p->knob.factor_sms;
    return need < cap ? need : cap;
}

template <int LOG2H>
static void run_row_fwd(sfft_plan *p, const double *img, const uint8_t *mask, cplx *inter, int NI, double *mu, int NMOM) {
    const Geom &g = p->g;
    const bool bulk = ((g.nx & 1) == 0) && (((size_t)img & 15) == 0);
    const int grid = row_grid<LOG2H>(p);
    const size_t sm = RowCfg<LOG2H>::SMEM_F;
    if (bulk && !mask) row_fwd_kernel<LOG2H, true, false><<<grid, ROW_THREADS, sm, p->stream>>>(img, mask, inter, NI, mu, NMOM, g, p->tw, p->rtw);
    else if (bulk) row_fwd_kernel<LOG2H, true, true><<<grid, ROW_THREADS, sm, p->stream>>>(img, mask, inter, NI, mu, NMOM, g, p->tw, p->rtw);
    else if (!mask) row_fwd_kernel<LOG2H, false, false><<<grid, ROW_THREADS, sm, p->stream>>>(img, mask, inter, NI, mu, NMOM, g, p->tw, p->rtw);
    else row_fwd_kernel<LOG2H, false, true><<<grid, ROW_THREADS, sm, p->stream>>>(img, mask, inter, NI, mu, NMOM, g, p->tw, p->rtw);
}

cudaError_t launch_row_fwd(sfft_plan *p, const double *img, const uint8_t *mask, cplx *inter, int NI, double *mu, int NMOM) {
    KLaunch kl(p, NI > 1 ? "row_fwd_R" : "row_fwd_S");
    switch (p->g.log2Hx) {
    case 9: run_row_fwd<9>(p, img, mask, inter, NI, mu, NMOM); break;
    case 10: run_row_fwd<10>(p, img, mask, inter, NI, mu, NMOM); break;
    case 11: run_row_fwd<11>(p, img, mask, inter, NI, mu, NMOM); break;
    default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

// inter must be the plan's intermediate buffer (the tensor map is built over it)
cudaError_t launch_row_inv(sfft_plan *p, const cplx *inter, const double *S, const double *coef, double *D, int mode) {
    const Geom &g = p->g;
    if (inter != p->inter) return cudaErrorInvalidValue;
    KLaunch kl(p, "row_inv");
    switch (g.log2Hx) {
    case 9: row_inv_kernel<9><<<row_grid<9>(p), ROW_THREADS, RowCfg<9>::XBYTES, p->stream>>>(*p->mapI, inter, S, coef, D, g, p->tw, mode); break;
    case 10: row_inv_kernel<10><<<row_grid<10>(p), ROW_THREADS, RowCfg<10>::XBYTES, p->stream>>>(*p->mapI, inter, S, coef, D, g, p->tw, mode); break;
    case 11: row_inv_kernel<11><<<row_grid<11>(p), ROW_THREADS, RowCfg<11>::XBYTES, p->stream>>>(*p->mapI, inter, S, coef, D, g, p->tw, mode); break;
    default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

} // namespace sfft
