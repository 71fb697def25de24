// sfft_cols.cu -- the column passes of the 2-D FFTs (steps a1 and a5; BASELINE.json north_star (a), (d); SURVEY.md
// 8(a) rows a1, a5): they move most of the path's bytes.
//
// Planes are column-major (sfft_fft.cuh: plane_idx), so a column is one contiguous run of My complex numbers.
// A WORKER is a group of T = My/16 threads that owns one column at a time: 16 values per thread in registers,
// radix-16 Stockham passes exchanged through the worker's own 16 My-byte shared-memory buffer (XOR-swizzled, no
// padding), synchronised by a named barrier of its own.  A CTA holds 256/T workers and two CTAs share an SM, so
// one worker's butterflies overlap another's exchanges and memory waits (a single 512-thread CTA per SM serialised
// them: profiles/r01l_ncu_summary.md).  Columns arrive quarter by quarter through a 3-slot ring of bulk
// global->shared copies (cp.async.bulk, SASS UBLKCP) that complete on mbarriers: one elected thread issues them,
// no per-thread copy instructions or address registers, and the copies of the next column are in flight while
// this one is transformed.  Results leave from the registers as 16-byte stores that are contiguous along ky
// (512 B per warp and instruction).
//
//   forward:  spec_k = FFT_y( yt^jj[k] * inter_ii[k] )       (one source column feeds all its jj's; re-read from L2)
//             column 0 of the intermediates is packed (X[0] + i X[Hx], both real along x): its transform F is
//             separated once, here, into the true columns kx = 0 and kx = Hx of the spectrum,
//                 F0[ky] = (F[ky] + conj F[-ky])/2,   FH[ky] = (F[ky] - conj F[-ky])/(2i),
//             so that every consumer sees Hx + 1 ordinary columns.
//   inverse:  inter = IFFT_y( sum_t spec_t * K^_t ),  K^_t at the thread's rows jrow + q1 My/4 (q1 < 4) from a 4-point
//             DFT of the L phase-shifted taps (khat4); column 0 is re-packed: M(kx=0) + i M(kx=Hx).
#include "sfft_internal.h"

namespace sfft {

constexpr int COL_THREADS = 256;
constexpr int COL_RING = 3;

template <int LOG2N> struct ColCfg {
    static constexpr int N = 1 << LOG2N, T = N / 16, G = COL_THREADS / T, QE = N / 4;
    static constexpr int R3 = N / 256;                       // radix of the third pass (2, 4, 8 or 16)
    static constexpr size_t SMEM = (size_t)G * N * sizeof(cplx) + (size_t)G * COL_RING * QE * sizeof(cplx);
};

// forward transform of the canonical registers (three passes, two exchanges); natural order on return
// after_x() is called once the thread has done its last read of X (the forward kernel hands X to the copy engine there)
template <int LOG2N, int DIR, typename F>
__device__ __forceinline__ void col_fft(cplx (&v)[16], cplx *X, int j, int bar_id, const cplx *__restrict__ tw, int Nt, cplx w2, cplx w3,
                                        F &&after_x) {
    using C = ColCfg<LOG2N>;
    constexpr int T = C::T;
    {   // pass 1: radix 16, no twiddles
        cplx x[16];
#pragma unroll
        for (int m = 0; m < 16; m++) x[m] = v[m];
        dft16<DIR>(x);
#pragma unroll
        for (int m = 0; m < 16; m++) X[out_pos<16, 4>(j, m, 0)] = x[m];
    }
    group_sync(bar_id, T);
    load_canonical<4, 1>(v, X, 0, j, T);
    group_sync(bar_id, T);
    {   // pass 2: radix 16, Ns = 16; one butterfly per thread, its twiddle lives in a register
        cplx x[16];
#pragma unroll
        for (int m = 0; m < 16; m++) x[m] = v[m];
        bfly_w<16, DIR>(x, w2);
#pragma unroll
        for (int m = 0; m < 16; m++) X[out_pos<16, 4>(j, m, 4)] = x[m];
    }
    group_sync(bar_id, T);
    load_canonical<4, 1>(v, X, 0, j, T);
    after_x();
    if (C::R3 == 16) {
        cplx x[16];
#pragma unroll
        for (int m = 0; m < 16; m++) x[m] = v[m];
        bfly_w<16, DIR>(x, w3);
#pragma unroll
        for (int m = 0; m < 16; m++) v[m] = x[m];
    } else {
        pass_regs<C::R3, DIR>(v, j, T, 8, tw, Nt);
    }
}

// ------------------------------------------------------------------------------------------ forward
// grid: persistent, <= 2 CTAs per SM; block 256 = G workers of T threads; dynamic smem ColCfg::SMEM.
// jobs packed 4 bits each, (ii << 2) | jj: output k = FFT_y(yt^jj * inter[ii]).
template <int LOG2N, typename ST>
__global__ void __launch_bounds__(COL_THREADS, 2)
col_fwd_kernel(const cplx *__restrict__ inter, ST *__restrict__ spec, unsigned long long jpack, int njobs, Geom g,
               const cplx *__restrict__ tw) {
    using C = ColCfg<LOG2N>;
    constexpr int N = C::N, T = C::T, G = C::G, QE = C::QE;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ unsigned long long full[G * 4], done[G * 4];
    const int grp = threadIdx.x / T, j = threadIdx.x - grp * T, bar_id = 1 + grp;
    cplx *X = reinterpret_cast<cplx *>(smem_raw) + (size_t)grp * N;
    cplx *ring = reinterpret_cast<cplx *>(smem_raw) + (size_t)G * N + (size_t)grp * COL_RING * QE;
    // FOUR landing slots, one per quarter of a column: quarters 0..2 in the ring, quarter 3 in the first quarter of the
    // exchange buffer X, which is idle from the last read of a transform to the first store of the next.  With three
    // slots the fourth quarter of a column could only be asked for when its first quarter had been consumed, and every
    // column waited a full memory latency for it (9-16 % of the kernel's stall samples sat on that wait).
    unsigned long long *bar = full + grp * 4, *rel = done + grp * 4;
    if (j == 0) {
        for (int s = 0; s < 4; s++) { mbar_init(&bar[s], 1); mbar_init(&rel[s], T); }
        mbar_fence_init();
    }
    __syncthreads();
    const int Hx = g.Hx, ny = g.ny, Nt = g.Nt;
    const int wid = blockIdx.x * G + grp, nw = gridDim.x * G;
    const int ncol = wid < Hx ? (Hx - wid + nw - 1) / nw : 0;
    const int nitems = ncol * njobs;
    const size_t iplane = (size_t)Hx * N, splane = (size_t)(Hx + 1) * N;
    const double inv_ny = 1.0 / (double)ny;
    auto slot_ptr = [&](int Q) -> cplx * { return Q < 3 ? ring + (size_t)Q * QE : X; };
    auto issue = [&](int n, int Q) { // one thread: quarter Q of item n into slot Q
        const int col = wid + (n / njobs) * nw, k = n % njobs;
        const int ii = (int)(jpack >> (4 * k + 2)) & 3;
        int rows = ny - Q * QE; rows = rows < 0 ? 0 : (rows > QE ? QE : rows);
        mbar_expect(&bar[Q], (unsigned)rows * 16u);
        if (rows > 0) bulk_g2s(slot_ptr(Q), inter + (size_t)ii * iplane + (size_t)col * N + Q * QE, (unsigned)rows * 16u, &bar[Q]);
    };
    if (j == 0 && nitems > 0)
        for (int Q = 0; Q < 4; Q++) issue(0, Q);
    const cplx w2 = tw[(size_t)(j & 15) * (Nt >> 8)];
    const cplx w3 = C::R3 == 16 ? tw[(size_t)(j & 255) * (Nt >> 12)] : mk(1.0, 0.0);
    const int j_outer_ = j; // (see the note at opaque_index)
    for (int n = 0; n < nitems; n++) {
        const int j = opaque_index(j_outer_);
        const int col = wid + (n / njobs) * nw, k = n % njobs;
        const int jp = (int)(jpack >> (4 * k)) & 3;
        const unsigned par = (unsigned)n & 1u;   // every slot is used once per item
        const bool more = n + 1 < nitems;
        // weight yt^jp as the one-hot cubic c0 + y (c1 + y (c2 + y c3)): three fused multiply-adds per row, no branches on jp
        const double c0 = jp == 0 ? 1.0 : 0.0, c1 = jp == 1 ? 1.0 : 0.0, c2 = jp == 2 ? 1.0 : 0.0, c3 = jp == 3 ? 1.0 : 0.0;
        const double y0 = (2.0 * j + 1.0 - ny) * inv_ny, ystep = 2.0 * T * inv_ny;
        cplx v[16];
#pragma unroll
        for (int Q = 0; Q < 4; Q++) {
            const cplx *src = Q < 3 ? ring + (size_t)Q * QE : X;
            mbar_wait(&bar[Q], par);
#pragma unroll
            for (int qq = 0; qq < 4; qq++) {
                const int q = 4 * Q + qq, row = j + T * q;
                cplx a = src[qq * T + j];
                const double yt = fma((double)q, ystep, y0);          // yt of row j + q T
                const double wgt = fma(yt, fma(yt, fma(yt, c3, c2), c1), c0);
                v[q] = row < ny ? cscale(a, wgt) : mk(0.0, 0.0);
            }
            // release the slot: every thread arrives (release semantics: its loads of the slot are done) and the issuing
            // thread refills it once all have.  (A bar.sync is not enough here: the copy engine is not ordered behind
            // it -- a refill could overtake a slow warp's reads.)  Slot 3 is X: it is busy until the transform's last read.
            if (Q < 3) {
                slot_release(&rel[Q]);
                if (j == 0 && more) { mbar_wait(&rel[Q], par); issue(n + 1, Q); }
            }
        }
        group_sync(bar_id, T); // quarter 3 has been read out of X by everyone (and so have the previous item's results)
        auto x_free = [&]() { // X goes to the copy engine: quarter 3 of the next item
            slot_release(&rel[3]);
            if (j == 0 && more) { mbar_wait(&rel[3], par); issue(n + 1, 3); }
        };
        ST *dst = spec + (size_t)k * splane;
        col_fft<LOG2N, -1>(v, X, j, bar_id, tw, Nt, w2, w3, [&] { if (col != 0) x_free(); });
        if (col != 0) {
#pragma unroll
            for (int q = 0; q < 16; q++) st_c(&dst[(size_t)col * N + j + q * T], v[q]);
        } else {
            // packed column: separate F = F0 + i FH through the exchange buffer (natural order, mirror read)
            group_sync(bar_id, T);
#pragma unroll
            for (int q = 0; q < 16; q++) X[swz<4>(j + q * T)] = v[q];
            group_sync(bar_id, T);
#pragma unroll
            for (int q = 0; q < 16; q++) {
                const int row = j + q * T;
                const cplx m = X[swz<4>((N - row) & (N - 1))];
                st_c(&dst[row], mk(0.5 * (v[q].x + m.x), 0.5 * (v[q].y - m.y)));
                st_c(&dst[(size_t)Hx * N + row], mk(0.5 * (v[q].y + m.y), -0.5 * (v[q].x - m.x)));
            }
            x_free();
        }
    }
}

// ------------------------------------------------------------------------------------------ inverse
// K^ of one (t, column) at the 4 rows jrow + q1 N/4 (q1 < 4):
//   K^[jrow + q1 N/4] = sum_v (E[v] e^{-2 pi i jrow v/N}) e^{-2 pi i q1 v/4}  -- a 4-point DFT of the
// L phase-shifted taps binned by v mod 4.  taps e[l], l = v + w; p1 = exp(-2 pi i jrow/N); the phase of tap v
// is p1^v, built by repeated multiplication (v <= 10).
__device__ __forceinline__ void khat4(cplx (&kh)[4], const cplx *e, int w, cplx p1) {
    kh[0] = e[w];
    kh[1] = mk(0.0, 0.0); kh[2] = mk(0.0, 0.0); kh[3] = mk(0.0, 0.0);
    cplx p = mk(1.0, 0.0);
#pragma unroll
    for (int v = 1; v <= (MAX_L - 1) / 2; v++) {
        if (v <= w) {
            p = cmul(p, p1);                                                   // exp(-2 pi i jrow v/N)
            const cplx a = cmul(e[w + v], p), b = cmul(e[w - v], cconj(p));
            kh[v & 3] = cadd(kh[v & 3], a);
            kh[(4 - (v & 3)) & 3] = cadd(kh[(4 - (v & 3)) & 3], b);
        }
    }
    dft4<-1>(kh[0], kh[1], kh[2], kh[3]);
}

// grid / block / smem as the forward kernel.  spec: NK planes of (Hx+1) columns; Ep: taps [NK][L][Hx+1];
// inter: one plane of Hx columns (rows < ny written).
template <int LOG2N, typename ST>
__global__ void __launch_bounds__(COL_THREADS, 2)
col_inv_kernel(const ST *__restrict__ spec, const cplx *__restrict__ Ep, cplx *__restrict__ inter, Geom g,
               const cplx *__restrict__ tw) {
    using C = ColCfg<LOG2N>;
    constexpr int N = C::N, T = C::T, G = C::G, QE = C::QE;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ unsigned long long full[G * COL_RING], done[G * COL_RING];
    const int grp = threadIdx.x / T, j = threadIdx.x - grp * T, bar_id = 1 + grp;
    cplx *X = reinterpret_cast<cplx *>(smem_raw) + (size_t)grp * N;
    cplx *ring = reinterpret_cast<cplx *>(smem_raw) + (size_t)G * N + (size_t)grp * COL_RING * QE;
    unsigned long long *bar = full + grp * COL_RING, *rel = done + grp * COL_RING;
    if (j == 0) {
        for (int s = 0; s < COL_RING; s++) { mbar_init(&bar[s], 1); mbar_init(&rel[s], T); }
        mbar_fence_init();
    }
    __syncthreads();
    const int Hx = g.Hx, ny = g.ny, Nt = g.Nt, L = g.L, w = g.w, NK = g.NK;
    const int wid = blockIdx.x * G + grp, nw = gridDim.x * G;
    const int ncol = wid < Hx ? (Hx - wid + nw - 1) / nw : 0;
    const size_t splane = (size_t)(Hx + 1) * N;
    // steps: per column nv = NK (2 NK for the packed column 0: its kx = 0 and kx = Hx parts) virtual spectra x 4 row sets
    const int nsteps = ncol > 0 ? 4 * (NK * ncol + (wid == 0 ? NK : 0)) : 0;
    int pn = 0, pv = 0, pq = 0, ps = 0; // producer cursor: column index, virtual spectrum, row set, step
    auto issue = [&]() {   // one thread: row set pq (rows T pq + 4T q1 + [0,T)) of virtual spectrum pv of column pn
        const int col = wid + pn * nw, nv = col == 0 ? 2 * NK : NK;
        const int t = pv % NK, sc = pv < NK ? col : Hx, slot = ps % COL_RING;
        const ST *src = spec + (size_t)t * splane + (size_t)sc * N + T * pq;
        mbar_expect(&bar[slot], (unsigned)(QE * sizeof(ST)));
#pragma unroll
        for (int q1 = 0; q1 < 4; q1++) bulk_g2s(reinterpret_cast<ST *>(ring + (size_t)slot * QE) + q1 * T, src + q1 * QE, (unsigned)(T * sizeof(ST)), &bar[slot]);
        ps++;
        if (++pq == 4) { pq = 0; if (++pv == nv) { pv = 0; pn++; } }
    };
    if (j == 0)
        for (int s = 0; s < COL_RING && s < nsteps; s++) issue();
    const cplx w2 = tw[(size_t)(j & 15) * (Nt >> 8)];
    const cplx w3 = C::R3 == 16 ? tw[(size_t)(j & 255) * (Nt >> 12)] : mk(1.0, 0.0);
    const int twsy = Nt / N;
    int s = 0;
    const int j_outer_ = j; // (see the note at opaque_index)
    for (int n = 0; n < ncol; n++) {
        const int j = opaque_index(j_outer_);
        const int col = wid + n * nw, nv = col == 0 ? 2 * NK : NK;
        group_sync(bar_id, T); // the previous column's last exchange has been read: X is free for the taps
        for (int e = j; e < nv * L; e += T) {
            const int vs = e / L, l = e - vs * L, t = vs % NK;
            X[e] = Ep[((size_t)t * L + l) * (Hx + 1) + (vs < NK ? col : Hx)];
        }
        group_sync(bar_id, T);
        cplx acc[16];
#pragma unroll
        for (int q = 0; q < 16; q++) acc[q] = mk(0.0, 0.0);
        for (int vs = 0; vs < nv; vs++) {
#pragma unroll
            for (int q0 = 0; q0 < 4; q0++, s++) {
                const int slot = s % COL_RING;
                cplx kh[4];
                khat4(kh, X + (size_t)vs * L, w, tw[(size_t)(j + T * q0) * twsy]);
                if (vs >= NK) {  // the kx = Hx part of the packed column enters as i * M
#pragma unroll
                    for (int q1 = 0; q1 < 4; q1++) kh[q1] = mk(-kh[q1].y, kh[q1].x);
                }
                mbar_wait(&bar[slot], (unsigned)(s / COL_RING) & 1u);
#pragma unroll
                for (int q1 = 0; q1 < 4; q1++) {
                    const cplx z = ld_c(reinterpret_cast<const ST *>(ring + (size_t)slot * QE)[q1 * T + j]);
                    cplx &a = acc[q0 + 4 * q1];
                    a.x = fma(z.x, kh[q1].x, fma(-z.y, kh[q1].y, a.x));
                    a.y = fma(z.x, kh[q1].y, fma(z.y, kh[q1].x, a.y));
                }
                slot_release(&rel[slot]); // release the slot (see col_fwd_kernel)
                if (j == 0 && s + COL_RING < nsteps) { mbar_wait(&rel[slot], (unsigned)(s / COL_RING) & 1u); issue(); }
            }
        }
        group_sync(bar_id, T); // every thread has read its taps from X
        col_fft<LOG2N, 1>(acc, X, j, bar_id, tw, Nt, w2, w3, [] {});
        cplx *dst = inter + (size_t)col * N;
#pragma unroll
        for (int q = 0; q < 16; q++) {
            const int row = j + q * T;
            if (row < ny) dst[row] = acc[q];
        }
    }
}

// plain kernel row tables Ep[t][v+w][kx] = sum_u a_{t,u,v} exp(-2 pi i kx u/Mx), kx = 0..Hx.
// grid = (ceil((Hx+1)/128), L, NK); block 128
__global__ void __launch_bounds__(128) ktab_plain_kernel(const double *__restrict__ coef, cplx *__restrict__ Ep, Geom g,
                                                        const cplx *__restrict__ tw) {
    const int kx = blockIdx.x * blockDim.x + threadIdx.x;
    if (kx > g.Hx) return;
    const int l = blockIdx.y, t = blockIdx.z, L = g.L, w = g.w, Mx = g.Mx;
    const double *a = coef + (size_t)t * L * L + (size_t)l * L + w; // a_{t,u,v} at a[u]
    cplx acc = mk(0.0, 0.0);
    for (int u = -w; u <= w; u++) {
        const cplx e = tw[(size_t)((kx * (u + Mx)) & (Mx - 1)) * (g.Nt / Mx)];
        acc.x = fma(a[u], e.x, acc.x); acc.y = fma(a[u], e.y, acc.y);
    }
    Ep[((size_t)t * L + l) * (g.Hx + 1) + kx] = acc;
}

// ------------------------------------------------------------------------------------------ host side
template <int LOG2N> static cudaError_t cols_attr() {
    cudaError_t e = cudaFuncSetAttribute(col_fwd_kernel<LOG2N, cplx>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ColCfg<LOG2N>::SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(col_fwd_kernel<LOG2N, float2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ColCfg<LOG2N>::SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(col_inv_kernel<LOG2N, cplx>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ColCfg<LOG2N>::SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(col_inv_kernel<LOG2N, float2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ColCfg<LOG2N>::SMEM);
    return e;
}
cudaError_t cols_init() { // per device, at plan creation
    cudaError_t e = cols_attr<9>();
    if (e == cudaSuccess) e = cols_attr<10>();
    if (e == cudaSuccess) e = cols_attr<11>();
    if (e == cudaSuccess) e = cols_attr<12>();
    return e;
}

static int col_grid(const sfft_plan *p, int reserve) {
    const Geom &g = p->g;
    const int G = COL_THREADS / (g.My / 16);
    int grid = 2 * p->sms;
    // while a factorisation runs beside us, leave a few SMs to it: a persistent CTA would otherwise block its chain
    // of small launches for the whole kernel
    if (reserve > 0 && grid > 2 * reserve) grid -= 2 * reserve;
    const int need = (g.Hx + G - 1) / G;
    return grid < need ? grid : need;
}

template <int LOG2N>
static void run_col_fwd(sfft_plan *p, int grid, const cplx *inter, void *spec, unsigned long long jpack, int ns) {
    if (p->spec32) col_fwd_kernel<LOG2N, float2><<<grid, COL_THREADS, ColCfg<LOG2N>::SMEM, p->stream>>>(inter, (float2 *)spec, jpack, ns, p->g, p->tw);
    else col_fwd_kernel<LOG2N, cplx><<<grid, COL_THREADS, ColCfg<LOG2N>::SMEM, p->stream>>>(inter, (cplx *)spec, jpack, ns, p->g, p->tw);
}
template <int LOG2N>
static void run_col_inv(sfft_plan *p, int grid, const void *spec, cplx *inter) {
    if (p->spec32) col_inv_kernel<LOG2N, float2><<<grid, COL_THREADS, ColCfg<LOG2N>::SMEM, p->stream>>>((const float2 *)spec, p->E, inter, p->g, p->tw);
    else col_inv_kernel<LOG2N, cplx><<<grid, COL_THREADS, ColCfg<LOG2N>::SMEM, p->stream>>>((const cplx *)spec, p->E, inter, p->g, p->tw);
}

// spec: ns planes of (Hx+1) x My spectrum elements (cplx, or float2 in the FP32-spectra plan mode)
cudaError_t launch_col_fwd(sfft_plan *p, const cplx *inter, void *spec, int ns, const int *ii, const int *jj) {
    const Geom &g = p->g;
    unsigned long long jpack = 0; // job k: (ii << 2) | jj, both <= 3 (DK <= 3)
    if (ns > 16) return cudaErrorInvalidValue;
    for (int k = 0; k < ns; k++) {
        if (ii[k] < 0 || ii[k] > 3 || jj[k] < 0 || jj[k] > 3) return cudaErrorInvalidValue;
        jpack |= (unsigned long long)((ii[k] << 2) | jj[k]) << (4 * k);
    }
    KLaunch kl(p, ns > 1 ? "col_fwd_R" : "col_fwd_S");
    const int grid = col_grid(p, p->factor_pending ? p->knob.factor_sms : 0);
    switch (g.log2My) {
    case 9: run_col_fwd<9>(p, grid, inter, spec, jpack, ns); break;
    case 10: run_col_fwd<10>(p, grid, inter, spec, jpack, ns); break;
    case 11: run_col_fwd<11>(p, grid, inter, spec, jpack, ns); break;
    case 12: run_col_fwd<12>(p, grid, inter, spec, jpack, ns); break;
    default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

cudaError_t launch_col_inv(sfft_plan *p, const void *spec, const double *coef, cplx *inter) {
    const Geom &g = p->g;
    { KLaunch kl(p, "ktab"); ktab_plain_kernel<<<dim3((g.Hx + 1 + 127) / 128, g.L, g.NK), 128, 0, p->stream>>>(coef, p->E, g, p->tw); }
    KLaunch kl(p, "col_inv");
    const int grid = col_grid(p, 0);
    switch (g.log2My) {
    case 9: run_col_inv<9>(p, grid, spec, inter); break;
    case 10: run_col_inv<10>(p, grid, spec, inter); break;
    case 11: run_col_inv<11>(p, grid, spec, inter); break;
    case 12: run_col_inv<12>(p, grid, spec, inter); break;
    default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

} // namespace sfft
