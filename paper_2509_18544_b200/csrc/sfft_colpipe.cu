// sfft_colpipe.cu -- persistent, software-pipelined column transforms (steps a1 and a5) for
// 512 <= My <= 4096: the column passes of the 2-D FFTs, which move most of the path's bytes.
//
// One CTA per SM loops over column tiles of 2 adjacent columns (32 contiguous bytes per spectrum
// row).  T = My/8 threads; thread j owns rows j + q T (q = 0..7) of BOTH columns in registers
// (2 x 8 complex), so the twiddle factors of a butterfly are computed once for two transforms.
//   * loads: every thread cp.async's exactly the elements it will use itself into a ring of two
//     one-column slots (no barrier is needed on that data) -- the next chunk streams in while the
//     current tile is being transformed: HBM latency is hidden inside one CTA;
//   * butterflies: radix-8 Stockham passes in registers, exchanged one column at a time through a
//     single padded shared-memory column (68 KB), results stored from registers, 32 B per row.
// forward:  spec_k = FFT_y( yt^jj[k] * inter_ii[k] )  -- one source tile feeds all its jj's;
// inverse:  inter = IFFT_y( sum_t spec_t * K^_t ),  K^_t at the thread's 8 rows from ONE 8-point DFT of
//           the L phase-shifted taps (K^_t[j + qT] = sum_v (E_t[v] e^{-2 pi i j v/My}) e^{-2 pi i q v/8}).
#include <cstdlib>
#include "sfft_internal.h"

namespace sfft {

constexpr int CP_E = 8;
constexpr int CP_MAXT = 512;

__device__ __forceinline__ void cpa16(void *smem_dst, const void *gsrc, bool valid) {
    const unsigned sa = (unsigned)__cvta_generic_to_shared(smem_dst);
    const int sz = valid ? 16 : 0; // src-size 0: zero fill
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(sa), "l"(gsrc), "r"(sz));
}
__device__ __forceinline__ void cpa_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N> __device__ __forceinline__ void cpa_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

__device__ __forceinline__ double ipw3(double b, int e) { double r = 1.0; for (int k = 0; k < e; k++) r *= b; return r; }

// Half-tile chunk h (rows j + q T with q = 2 qq + h, qq < 4, both columns) into slot[(qq*T + j)*2 + col].
// Lanes 2k, 2k+1 copy the two 16-byte halves of the SAME 32-byte row segment (first the even lane's
// row, then the odd lane's), so a warp request covers whole sectors; the data of a thread is copied
// by itself and its lane partner: cpa_wait + __syncwarp() make it visible, no CTA barrier.
// rs = row stride of the source in complex elements (Hx for the row-major intermediates, 2 for tile-major spectra)
__device__ __forceinline__ void chunk_issue(cplx *slot, const cplx *tile_src, int h, int rs, int nrows, int j, int T) {
    const int col = j & 1;
#pragma unroll
    for (int qq = 0; qq < CP_E / 2; qq++) {
#pragma unroll
        for (int o = 0; o < 2; o++) {
            const int jo = (j & ~1) | o, row = jo + (2 * qq + h) * T;
            const bool ok = row < nrows;
            cpa16(slot + (size_t)(qq * T + jo) * 2 + col, ok ? tile_src + (size_t)row * rs + col : tile_src, ok);
        }
    }
    cpa_commit();
}

// registers -> global, 32 contiguous bytes per lane pair and row (one shuffle per value)
__device__ __forceinline__ void store_pair(cplx *tile_dst, const cplx (&v)[2][CP_E], int rs, int nrows, int j, int T) {
    const bool odd = j & 1;
#pragma unroll
    for (int q = 0; q < CP_E; q++) {
        const cplx send = odd ? v[0][q] : v[1][q];
        cplx recv;
        recv.x = __shfl_xor_sync(0xffffffffu, send.x, 1);
        recv.y = __shfl_xor_sync(0xffffffffu, send.y, 1);
        const int rowA = (j & ~1) + q * T, rowB = rowA + 1;
        const cplx va = odd ? recv : v[0][q], vb = odd ? v[1][q] : recv;
        if (rowA < nrows) tile_dst[(size_t)rowA * rs + (odd ? 1 : 0)] = va;
        if (rowB < nrows) tile_dst[(size_t)rowB * rs + (odd ? 1 : 0)] = vb;
    }
}

// One radix-R pass over both columns; twiddles shared.  X: single-column padded scratch.
// STORE: exchange through X (column 0, then column 1); else results stay canonical in v.
// wpre: for radix-8 passes (one butterfly per thread) the pass twiddle exp(-2 pi i k/(8 Ns)), k = j mod Ns, is the
// same for every tile a thread transforms: it is loaded once per kernel and passed in (HAVEW).
template <int R, int DIR, bool STORE, bool HAVEW = false>
__device__ __forceinline__ void pass2(cplx (&v)[2][CP_E], cplx *X, int j, int T, int log2Ns, const cplx *tw, int Nt,
                                      cplx wpre = cplx()) {
    constexpr int NBF = CP_E / R;
    constexpr int LOG2R = (R == 8) ? 3 : (R == 4) ? 2 : 1;
    const int Ns = 1 << log2Ns;
#pragma unroll
    for (int c = 0; c < 2; c++) {
        if (STORE) __syncthreads(); // every thread has finished reading X
#pragma unroll
        for (int b = 0; b < NBF; b++) {
            cplx x[R];
#pragma unroll
            for (int m = 0; m < R; m++) x[m] = v[c][b + m * NBF];
            const int jb = j + b * T;
            const int k = jb & (Ns - 1);
            if (log2Ns > 0) {
                cplx w1 = HAVEW ? wpre : tw[(size_t)k * (Nt >> (log2Ns + LOG2R))];
                if (DIR > 0) w1.y = -w1.y;
                twiddle_powers<R>(x, w1);
            }
            dftR<R, DIR>(x);
            if (STORE) {
                const int base = ((jb >> log2Ns) << (log2Ns + LOG2R)) + k;
#pragma unroll
                for (int m = 0; m < R; m++) X[padE<CP_E>(base + (m << log2Ns))] = x[m];
            } else {
#pragma unroll
                for (int m = 0; m < R; m++) v[c][b + m * NBF] = x[m];
            }
        }
        if (STORE) {
            __syncthreads();
#pragma unroll
            for (int q = 0; q < CP_E; q++) v[c][q] = X[padE<CP_E>(j + q * T)];
        }
    }
}

// twiddles of the radix-8 passes 2..4 of this thread (log2Ns = 3, 6, 9), loaded once per kernel
struct PassTw { cplx w[3]; };
__device__ __forceinline__ PassTw load_pass_tw(int log2N, int j, const cplx *tw, int Nt) {
    PassTw p;
#pragma unroll
    for (int k = 0; k < 3; k++) {
        const int log2Ns = 3 * (k + 1);
        p.w[k] = (log2Ns + 3 <= log2N) ? tw[(size_t)(j & ((1 << log2Ns) - 1)) * (Nt >> (log2Ns + 3))] : mk(1.0, 0.0);
    }
    return p;
}

// LOG2N_CT != 0: length fixed at compile time (My = 4096), all index arithmetic folds to constants.
// wsm (optional): the thread's pass twiddles parked in shared memory, wsm[pass * T + j] (the forward kernel has
// no registers to spare and almost no L1 left beside its 200 KB of shared memory).
template <int DIR, bool PW, int LOG2N_CT>
__device__ __forceinline__ void fft2col(cplx (&v)[2][CP_E], cplx *X, int log2N_rt, int j, const cplx *tw, int Nt, const PassTw &pw,
                                        const cplx *wsm = nullptr) {
    const int log2N = LOG2N_CT ? LOG2N_CT : log2N_rt;
    const int T = 1 << (log2N - 3);
    cplx wa = cplx();
    if (!PW && LOG2N_CT == 12 && !wsm) wa = tw[(size_t)(j & 7) * (Nt >> 6)];
    pass2<8, DIR, true>(v, X, j, T, 0, tw, Nt);
    if (LOG2N_CT) {
        if (wsm) {
            if (6 < log2N) pass2<8, DIR, true, true>(v, X, j, T, 3, tw, Nt, wsm[j]);
            if (9 < log2N) pass2<8, DIR, true, true>(v, X, j, T, 6, tw, Nt, wsm[T + j]);
            const int log2Ns = (9 < log2N) ? 9 : (6 < log2N) ? 6 : 3, ip = log2Ns / 3 - 1;
            switch (log2N - log2Ns) {
            case 3: pass2<8, DIR, false, true>(v, X, j, T, log2Ns, tw, Nt, wsm[ip * T + j]); break;
            case 2: pass2<4, DIR, false>(v, X, j, T, log2Ns, tw, Nt); break;
            default: pass2<2, DIR, false>(v, X, j, T, log2Ns, tw, Nt); break;
            }
            return;
        }
        if (!PW && LOG2N_CT == 12) {
            // no registers for resident pass twiddles (forward kernel): fetch the twiddle of pass k+1 BEFORE the
            // exchange of pass k, so that its L2 latency hides behind the barriers instead of stalling the butterflies
            const cplx wb = tw[(size_t)(j & 63) * (Nt >> 9)];
            pass2<8, DIR, true, true>(v, X, j, T, 3, tw, Nt, wa);
            const cplx wc = tw[(size_t)(j & 511) * (Nt >> 12)];
            pass2<8, DIR, true, true>(v, X, j, T, 6, tw, Nt, wb);
            pass2<8, DIR, false, true>(v, X, j, T, 9, tw, Nt, wc);
            return;
        }
        if (6 < log2N) pass2<8, DIR, true, PW>(v, X, j, T, 3, tw, Nt, pw.w[0]);
        if (9 < log2N) pass2<8, DIR, true, PW>(v, X, j, T, 6, tw, Nt, pw.w[1]);
        const int log2Ns = (9 < log2N) ? 9 : (6 < log2N) ? 6 : 3, ip = log2Ns / 3 - 1;
        switch (log2N - log2Ns) {
        case 3: pass2<8, DIR, false, PW>(v, X, j, T, log2Ns, tw, Nt, pw.w[ip]); break;
        case 2: pass2<4, DIR, false>(v, X, j, T, log2Ns, tw, Nt); break;
        default: pass2<2, DIR, false>(v, X, j, T, log2Ns, tw, Nt); break;
        }
        return;
    }
    int log2Ns = 3, ip = 0;
#pragma unroll
    for (int it = 0; it < 2; it++)
        if (log2Ns + 3 < log2N) { pass2<8, DIR, true, PW>(v, X, j, T, log2Ns, tw, Nt, pw.w[ip]); log2Ns += 3; ip++; }
    switch (log2N - log2Ns) {
    case 3: pass2<8, DIR, false, PW>(v, X, j, T, log2Ns, tw, Nt, pw.w[ip]); break;
    case 2: pass2<4, DIR, false>(v, X, j, T, log2Ns, tw, Nt); break;
    default: pass2<2, DIR, false>(v, X, j, T, log2Ns, tw, Nt); break;
    }
}

// ------------------------------------------------------------------------------------------ forward
// grid = min(#SM, Hx/2) persistent CTAs; block = My/8; dynamic smem = (padded_lenE<8>(My) + 2 My) cplx.
template <int LOG2N_CT>
__global__ void __launch_bounds__(CP_MAXT, 1)
colpipe_fwd_kernel(const cplx *__restrict__ inter, cplx *__restrict__ spec, unsigned long long jpack, int njobs, int nsrc, Geom g,
                   const cplx *__restrict__ tw) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int My = LOG2N_CT ? (1 << LOG2N_CT) : g.My, Hx = g.Hx, T = My / CP_E, j = threadIdx.x;
    cplx *X = reinterpret_cast<cplx *>(smem_raw);
    cplx *ring = X + padded_lenE<CP_E>(My);
    const int ntiles = Hx / 2;
    const int my_tiles = (ntiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
    const int nitems = my_tiles * nsrc;
    const size_t src_plane = (size_t)g.ny * Hx, plane = (size_t)My * Hx;
    const double inv_ny = 1.0 / (double)g.ny;
    const PassTw pw = PassTw();
    const cplx *wsm = nullptr; // (parking the pass twiddles in shared memory measured slower than the L1/L2 loads)
    auto issue_item = [&](int n) {
        if (n < nitems) {
            const int tile = blockIdx.x + (n / nsrc) * gridDim.x, i = n % nsrc;
            const cplx *src = inter + (size_t)i * src_plane + 2 * tile;
            chunk_issue(ring, src, 0, Hx, g.ny, j, T);
            chunk_issue(ring + My, src, 1, Hx, g.ny, j, T);
        } else { cpa_commit(); cpa_commit(); }
    };
    issue_item(0);
    for (int n = 0; n < nitems; n++) {
        const int tile = blockIdx.x + (n / nsrc) * gridDim.x, i = n % nsrc;
        // jobs packed 4 bits each, (ii << 2) | jj, in a register: no table look-ups on the critical path
        int last = -1;
        for (int k = 0; k < njobs; k++) if ((int)((jpack >> (4 * k + 2)) & 3) == i) last = k;
        cpa_wait<0>();
        __syncwarp();
        for (int k = 0; k < njobs; k++) {
            const int jb = (int)(jpack >> (4 * k)) & 15;
            if ((jb >> 2) != i) continue;
            const int jp = jb & 3;
            cplx v[2][CP_E];
#pragma unroll
            for (int q = 0; q < CP_E; q++) {
                const double wgt = jp > 0 ? ipw3((2.0 * (j + q * T) + 1.0 - g.ny) * inv_ny, jp) : 1.0;
                const cplx *e = ring + (size_t)(q & 1) * My + (size_t)((q >> 1) * T + j) * 2;
                v[0][q] = cscale(e[0], wgt);
                v[1][q] = cscale(e[1], wgt);
            }
            if (k == last) { __syncwarp(); issue_item(n + 1); } // both lanes of a pair have read: the slots are free
            fft2col<-1, false, LOG2N_CT>(v, X, g.log2My, j, tw, g.Nt, pw, wsm);
            store_pair(spec + (size_t)k * plane + (size_t)tile * My * 2, v, 2, My, j, T);
        }
    }
    cpa_wait<0>();
}

// ------------------------------------------------------------------------------------------ inverse
// K^ of one (t, column) at the 4 rows jrow + 2 q' T (q' < 4) of a thread (jrow = j + h T):
//   K^[jrow + 2 q' T] = sum_v (E[v] e^{-2 pi i jrow v/My}) e^{-2 pi i q' v/4}  -- a 4-point DFT of the
// L phase-shifted taps binned by v mod 4.  taps e[l * estride], l = v + w; phases from tw.
// p1 = exp(-2 pi i jrow/My); the phase of tap v is p1^v, built by repeated multiplication (v <= 10).
__device__ __forceinline__ void khat4(cplx (&kh)[4], const cplx *e, int estride, int w, cplx p1) {
    kh[0] = e[w * estride];
    kh[1] = mk(0.0, 0.0); kh[2] = mk(0.0, 0.0); kh[3] = mk(0.0, 0.0);
    cplx p = mk(1.0, 0.0);
#pragma unroll
    for (int v = 1; v <= (MAX_L - 1) / 2; v++) {
        if (v <= w) {
            p = cmul(p, p1);                                                   // exp(-2 pi i jrow v/My)
            const cplx a = cmul(e[(w + v) * estride], p), b = cmul(e[(w - v) * estride], cconj(p));
            kh[v & 3] = cadd(kh[v & 3], a);
            kh[(4 - (v & 3)) & 3] = cadd(kh[(4 - (v & 3)) & 3], b);
        }
    }
    dft4<-1>(kh[0], kh[1], kh[2], kh[3]);
}

// grid = min(#SM, Hx/2); block = My/8; dynamic smem = (padded_lenE<8>(My) + 2 My + 3 NK L) cplx.
// Ep: plain taps [NK][L][Hx+1].
template <int LOG2N_CT>
__global__ void __launch_bounds__(CP_MAXT, 1)
colpipe_inv_kernel(const cplx *__restrict__ spec, const cplx *__restrict__ Ep, cplx *__restrict__ inter, Geom g,
                   const cplx *__restrict__ tw) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int My = LOG2N_CT ? (1 << LOG2N_CT) : g.My, Hx = g.Hx, T = My / CP_E, j = threadIdx.x, L = g.L, w = g.w, NK = g.NK;
    cplx *X = reinterpret_cast<cplx *>(smem_raw);
    cplx *ring = X + padded_lenE<CP_E>(My);
    cplx *et = ring + 2 * My; // [t*L + l][3]: columns 0, 1 of the tile; slot 2: second tap set of the packed column
    const int ntiles = Hx / 2;
    const int my_tiles = (ntiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
    const int nchunks = my_tiles * NK * 2;
    const size_t plane = (size_t)My * Hx;
    const int twsy = g.Nt / My;
    const PassTw pw = load_pass_tw(g.log2My, j, tw, g.Nt);
    const cplx ph1[2] = {tw[(size_t)j * twsy], tw[(size_t)(j + T) * twsy]}; // exp(-2 pi i (j + h T)/My), h = 0, 1
    auto issue_chunk = [&](int s) { // chunk s = ((tile index * NK) + t) * 2 + h  ->  slot h
        if (s < nchunks) {
            const int tile = blockIdx.x + (s / (2 * NK)) * gridDim.x, t = (s >> 1) % NK, h = s & 1;
            chunk_issue(ring + h * My, spec + (size_t)t * plane + (size_t)tile * My * 2, h, 2, My, j, T);
        } else cpa_commit();
    };
    issue_chunk(0); issue_chunk(1);
    for (int it = 0; it < my_tiles; it++) {
        const int tile = blockIdx.x + it * gridDim.x;
        __syncthreads(); // previous tile's readers of et are done
        for (int e = j; e < NK * L * 3; e += T) {
            const int cc = e % 3, sl = e / 3;
            const cplx *row = Ep + (size_t)sl * (Hx + 1);
            cplx val;
            if (tile == 0 && cc != 1) { // packed column: Z K0' + conj(Zm) K0'',  K0' = (K(0)+K(Hx))/2, K0'' = (K(0)-K(Hx))/2
                const cplx e0 = row[0], eH = row[Hx];
                val = cc == 0 ? mk(0.5 * (e0.x + eH.x), 0.5 * (e0.y + eH.y)) : mk(0.5 * (e0.x - eH.x), 0.5 * (e0.y - eH.y));
            } else val = cc < 2 ? row[2 * tile + cc] : mk(0.0, 0.0);
            et[e] = val;
        }
        __syncthreads();
        cplx acc[2][CP_E];
#pragma unroll
        for (int q = 0; q < CP_E; q++) { acc[0][q] = mk(0.0, 0.0); acc[1][q] = mk(0.0, 0.0); }
        for (int t = 0; t < NK; t++) {
#pragma unroll
            for (int h = 0; h < 2; h++) {
                const int s = (it * NK + t) * 2 + h;
                cplx k0[4], k1[4];
                khat4(k0, et + (size_t)t * L * 3 + 0, 3, w, ph1[h]);
                khat4(k1, et + (size_t)t * L * 3 + 1, 3, w, ph1[h]);
                cpa_wait<1>();
                __syncwarp();
                const cplx *slot = ring + h * My;
#pragma unroll
                for (int qq = 0; qq < 4; qq++) {
                    const cplx z0 = slot[(size_t)(qq * T + j) * 2], z1 = slot[(size_t)(qq * T + j) * 2 + 1];
                    cplx &a0 = acc[0][2 * qq + h], &a1 = acc[1][2 * qq + h];
                    a0.x = fma(z0.x, k0[qq].x, fma(-z0.y, k0[qq].y, a0.x));
                    a0.y = fma(z0.x, k0[qq].y, fma(z0.y, k0[qq].x, a0.y));
                    a1.x = fma(z1.x, k1[qq].x, fma(-z1.y, k1[qq].y, a1.x));
                    a1.y = fma(z1.x, k1[qq].y, fma(z1.y, k1[qq].x, a1.y));
                }
                __syncwarp();
                issue_chunk(s + 2);
                if (tile == 0) {
                    khat4(k0, et + (size_t)t * L * 3 + 2, 3, w, ph1[h]);
                    const cplx *zc = spec + (size_t)t * plane;
#pragma unroll
                    for (int qq = 0; qq < 4; qq++) {
                        const cplx z = cconj(zc[(size_t)((My - (j + (2 * qq + h) * T)) & (My - 1)) * 2]); // tile 0, column 0
                        cplx &a0 = acc[0][2 * qq + h];
                        a0.x = fma(z.x, k0[qq].x, fma(-z.y, k0[qq].y, a0.x));
                        a0.y = fma(z.x, k0[qq].y, fma(z.y, k0[qq].x, a0.y));
                    }
                }
            }
        }
        fft2col<1, true, LOG2N_CT>(acc, X, g.log2My, j, tw, g.Nt, pw);
        store_pair(inter + 2 * tile, acc, Hx, g.ny, j, T);
    }
    cpa_wait<0>();
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

bool colpipe_ok(const Geom &g) { return g.My >= 512 && g.My <= 4096 && g.Hx >= 2 && getenv("SFFT_NO_COLPIPE") == nullptr; }

static int colpipe_reserve() { const char *e = getenv("SFFT_FACTOR_SMS"); return e ? atoi(e) : 12; }
static int colpipe_grid(const Geom &g, int reserve) {
    static int sms = 0;
    if (!sms) { int dev = 0; cudaGetDevice(&dev); cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev); if (sms <= 0) sms = 148; }
    const int ntiles = g.Hx / 2;
    int grid = ntiles < sms ? ntiles : sms;
    // while a factorisation runs beside us, leave a few SMs to it: a persistent full-register CTA would
    // otherwise block its chain of small launches for the whole kernel
    if (reserve > 0 && grid > 4 * reserve) grid -= reserve;
    return grid;
}

cudaError_t launch_colpipe_fwd(sfft_plan *p, const cplx *inter, cplx *spec, int ns, const int *ii, const int *jj, int nsrc) {
    const Geom &g = p->g;
    const size_t smem = (size_t)(padded_lenE<CP_E>(g.My) + 2 * g.My + 0) * sizeof(cplx);
    static bool attr_set = false;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(colpipe_fwd_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, 220 * 1024);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(colpipe_fwd_kernel<12>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    unsigned long long jpack = 0; // job k: (ii << 2) | jj, both <= 3 (DK <= 3)
    for (int k = 0; k < ns; k++) {
        if (ii[k] < 0 || ii[k] > 3 || jj[k] < 0 || jj[k] > 3 || ns > 16) return cudaErrorInvalidValue;
        jpack |= (unsigned long long)((ii[k] << 2) | jj[k]) << (4 * k);
    }
    KLaunch kl(p, ns > 1 ? "col_fwd_R" : "col_fwd_S");
    const int grid = colpipe_grid(g, p->factor_pending ? colpipe_reserve() : 0);
    if (g.log2My == 12) colpipe_fwd_kernel<12><<<grid, g.My / CP_E, smem, p->stream>>>(inter, spec, jpack, ns, nsrc, g, p->tw);
    else colpipe_fwd_kernel<0><<<grid, g.My / CP_E, smem, p->stream>>>(inter, spec, jpack, ns, nsrc, g, p->tw);
    return cudaGetLastError();
}

cudaError_t launch_colpipe_inv(sfft_plan *p, const cplx *spec, const double *coef, cplx *inter) {
    const Geom &g = p->g;
    { KLaunch kl(p, "ktab"); ktab_plain_kernel<<<dim3((g.Hx + 1 + 127) / 128, g.L, g.NK), 128, 0, p->stream>>>(coef, p->E, g, p->tw); }
    const size_t smem = (size_t)(padded_lenE<CP_E>(g.My) + 2 * g.My + 3 * g.NK * g.L) * sizeof(cplx);
    static bool attr_set = false;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(colpipe_inv_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, 224 * 1024);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(colpipe_inv_kernel<12>, cudaFuncAttributeMaxDynamicSharedMemorySize, 224 * 1024);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    KLaunch kl(p, "col_inv");
    if (g.log2My == 12) colpipe_inv_kernel<12><<<colpipe_grid(g, 0), g.My / CP_E, smem, p->stream>>>(spec, p->E, inter, g, p->tw);
    else colpipe_inv_kernel<0><<<colpipe_grid(g, 0), g.My / CP_E, smem, p->stream>>>(spec, p->E, inter, g, p->tw);
    return cudaGetLastError();
}

} // namespace sfft
